// lbwp_convert.cuh -- external dense moments <-> internal ghost-padded deviation storage.
// Only lbwp_init / lbwp_set_moments / lbwp_moments use these; they are not on the
// per-step path.  The shifts are taken in fp64 and rounded once to the state type.
#pragma once
#include "lbwp_common.cuh"

namespace lbwp {

// ext: [M][nz][ny][nx] (include/lbwp.h)  ->  dst: internal fields incl. ghost images.
template <typename T, int NC>
__global__ void __launch_bounds__(256) k_import_moments(Layout L, const T* __restrict__ ext, T* __restrict__ dst) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const long long F = L.field;
    int ke = 0, ki = 0;
    if (NC == 1) {
        store_images(dst + (ki++) * F, L, x, y, z, T((double)ext[(ke++) * n + e] - 1.0));
    } else {
        const double ra = (double)ext[e], rb = (double)ext[n + e];
        ke = 2;
        store_images(dst + (ki++) * F, L, x, y, z, T(ra));
        store_images(dst + (ki++) * F, L, x, y, z, T((ra + rb) - 1.0));
    }
    for (int a = 0; a < 3; ++a) store_images(dst + (ki++) * F, L, x, y, z, ext[(ke++) * n + e]);
    for (int a = 0; a < 3; ++a)
        store_images(dst + (ki++) * F, L, x, y, z, T((double)ext[(ke++) * n + e] - 1.0 / 3.0));
    for (int a = 0; a < 3; ++a) store_images(dst + (ki++) * F, L, x, y, z, ext[(ke++) * n + e]);
}

template <typename T, int NC>
__global__ void __launch_bounds__(256) k_export_moments(Layout L, const T* __restrict__ src, T* __restrict__ ext) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const long long c = lidx(L, x, y, z);
    const long long F = L.field;
    int ke = 0, ki = 0;
    if (NC == 1) {
        ext[(ke++) * n + e] = T(1.0 + (double)src[(ki++) * F + c]);
    } else {
        const double ra = (double)src[c], rho = 1.0 + (double)src[F + c];
        ki = 2;
        ext[(ke++) * n + e] = T(ra);
        ext[(ke++) * n + e] = T(rho - ra);
    }
    for (int a = 0; a < 3; ++a) ext[(ke++) * n + e] = src[(ki++) * F + c];
    for (int a = 0; a < 3; ++a) ext[(ke++) * n + e] = T((double)src[(ki++) * F + c] + 1.0 / 3.0);
    for (int a = 0; a < 3; ++a) ext[(ke++) * n + e] = src[(ki++) * F + c];
}

}  // namespace lbwp
