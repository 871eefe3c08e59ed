// lbwp_common.cuh -- device-side layout and helpers shared by the sm_100a kernels.
//
// Internal state layout (private to the library; include/lbwp.h documents the
// external one).  Every field is a ghost-padded box
//     [pz = nz+2][py = ny+2][px]      x fastest,
// interior node (x,y,z) at ((z+1)*py + (y+1))*px + ox + x, one ghost cell on each
// side in every direction holding the periodic image (reading C13), so the step
// kernels never wrap an index.  ox = 32 bytes worth of elements and px is a
// multiple of 32 bytes, so interior rows start on a DRAM sector boundary.
// The writer of a boundary node also writes its ghost images (store_images), so
// no separate halo pass exists.
//
// Stored fields ("deviation storage"): the moments of
// PAPER.md:39 minus their rest-state values, which the linear part of the update
// reproduces exactly, so fp32 keeps ~7 digits of the *deviation*:
//   ncomp==1 (M=10): drho = rho-1, ux, uy, uz, dPxx = Pxx-1/3, dPyy, dPzz, Pxy, Pxz, Pyz
//   ncomp==2 (M=11): rhoA, drho = rhoA+rhoB-1, ux, uy, uz, dPxx, dPyy, dPzz, Pxy, Pxz, Pyz
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lbwp {

struct Layout {
    int nx, ny, nz;     // interior box
    int ox;             // x offset of interior node 0 inside a row
    int px, py, pz;     // padded extents
    long long plane;    // px*py
    long long field;    // px*py*pz elements per field
};

__host__ __device__ inline long long lidx(const Layout& L, int x, int y, int z) {
    return ((long long)(z + 1) * L.py + (y + 1)) * L.px + L.ox + x;
}

inline Layout make_layout(int nx, int ny, int nz, int elem_bytes) {
    Layout L;
    L.nx = nx; L.ny = ny; L.nz = nz;
    const int q = 32 / elem_bytes;               // elements per 32-byte sector
    L.ox = q;
    L.px = ((L.ox + nx + 1 + q - 1) / q) * q;
    L.py = ny + 2;
    L.pz = nz + 2;
    L.plane = (long long)L.px * L.py;
    L.field = L.plane * L.pz;
    return L;
}

// Scalars of one run, in the arithmetic type.
template <typename T>
struct StepParams {
    Layout L;
    const T* __restrict__ src;   // M fields, field stride L.field
    T* __restrict__ dst;
    const T* __restrict__ grad;  // ncomp==2: 3 fields Gx,Gy,Gz (same layout), else nullptr
    T omega;                     // 1/tau            (reading C3)
    T A, beta;                   // colour gradient  (reading C6)
    const T* __restrict__ force = nullptr;   // near-contact force Fx, Fy, Fz (same layout), or nullptr (readings C20-C24)
    T A_h = T(0), h_c = T(0);    // its strength and cut-off distance (Eq. 10)
};

// Store v at interior node (x,y,z) of one field and at each of its periodic ghost
// images (up to 7 more for a corner node of the box).
template <typename T>
__device__ __forceinline__ void store_images(T* __restrict__ f, const Layout& L, int x, int y, int z, T v) {
    const long long c = lidx(L, x, y, z);
    f[c] = v;
    const bool bx0 = (x == 0), bx1 = (x == L.nx - 1);
    const bool by0 = (y == 0), by1 = (y == L.ny - 1);
    const bool bz0 = (z == 0), bz1 = (z == L.nz - 1);
    if (!(bx0 | bx1 | by0 | by1 | bz0 | bz1)) return;
    // image offsets along each axis: none, +n (node at 0), -n (node at n-1); a box one node thick has both.
    // Plain selects, no indexed arrays: those would live in local memory and cost every caller stack traffic.
    const long long xs1 = bx0 ? (long long)L.nx : 0, xs2 = bx1 ? -(long long)L.nx : 0;
    const long long ys1 = by0 ? (long long)L.ny * L.px : 0, ys2 = by1 ? -(long long)L.ny * L.px : 0;
    const long long zs1 = bz0 ? (long long)L.nz * L.plane : 0, zs2 = bz1 ? -(long long)L.nz * L.plane : 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const long long dz = k == 0 ? 0 : k == 1 ? zs1 : zs2;
        if (k && !dz) continue;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const long long dy = j == 0 ? 0 : j == 1 ? ys1 : ys2;
            if (j && !dy) continue;
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                const long long dx = i == 0 ? 0 : i == 1 ? xs1 : xs2;
                if ((i && !dx) || i + j + k == 0) continue;
                f[c + dz + dy + dx] = v;
            }
        }
    }
}

// D3Q27 / D3Q19 weights by |c|^2 (textbook values; PAPER.md:58 leaves them to
// "the lattice geometry").  cs^2 = 1/3.
template <int Q>
__host__ __device__ constexpr double lattice_w(int n2) {
    return Q == 27 ? (n2 == 0 ? 8.0 / 27.0 : n2 == 1 ? 2.0 / 27.0 : n2 == 2 ? 1.0 / 54.0 : 1.0 / 216.0)
                   : (n2 == 0 ? 1.0 / 3.0 : n2 == 1 ? 1.0 / 18.0 : n2 == 2 ? 1.0 / 36.0 : 0.0);
}

template <typename T> __device__ __forceinline__ T rsqrt_t(T x);
template <> __device__ __forceinline__ float rsqrt_t<float>(float x) { return 1.0f / sqrtf(x); }
template <> __device__ __forceinline__ double rsqrt_t<double>(double x) { return 1.0 / sqrt(x); }

}  // namespace lbwp
