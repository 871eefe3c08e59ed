// lbwp_diag.cuh -- the paper's diagnostics as ONE fused reduction over the current moments (Fig. 2,
// 3, 5, 7): colour masses sum(rhoA), sum(rhoB), total momentum sum(rho u), the mean density of the dense phase
// <rho>_{rho > threshold} with its node count, the maximum density, and the densities at probe sites.
// "rho" of the paper's droplet figures is the density of the droplet component (its field ranges from 0 to 1,
// PAPER.md:118): rhoA for two-component runs, rho itself for single-component ones.
// Input: the dense external moments [M][nz][ny][nx] (lbwp_moments' layout) in device memory.  Sums are taken in fp64:
// each block reduces its slice, block partials land in a buffer, and the last pass adds them in a fixed order, so the
// result does not depend on scheduling.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lbwp {

constexpr int DIAG_NSUM = 8;       // rhoA, rhoB, jx, jy, jz, sum of rho above threshold, count above, (unused)
constexpr int DIAG_BLOCKS = 592;   // 4 per SM on 148 SMs
constexpr int DIAG_THREADS = 256;

template <typename T, int NC>
__global__ void __launch_bounds__(DIAG_THREADS) k_diag_partial(const T* __restrict__ m, long long n, double threshold,
                                                               double* __restrict__ partial /* [blocks][NSUM + 1] */) {
    double s[DIAG_NSUM] = {0, 0, 0, 0, 0, 0, 0, 0};
    double mx = -1e300;
    constexpr int off = NC - 1;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double ra = (double)m[i];
        const double rb = NC == 2 ? (double)m[n + i] : 0.0;
        const double rho = ra + rb;
        s[0] += ra;
        s[1] += rb;
        s[2] += rho * (double)m[(off + 1) * n + i];
        s[3] += rho * (double)m[(off + 2) * n + i];
        s[4] += rho * (double)m[(off + 3) * n + i];
        if (ra > threshold) { s[5] += ra; s[6] += 1.0; }
        mx = ra > mx ? ra : mx;
    }
    __shared__ double sh[DIAG_THREADS / 32][DIAG_NSUM + 1];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < DIAG_NSUM; ++k)
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) s[k] += __shfl_down_sync(0xffffffffu, s[k], d);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) { const double o = __shfl_down_sync(0xffffffffu, mx, d); mx = o > mx ? o : mx; }
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < DIAG_NSUM; ++k) sh[w][k] = s[k];
        sh[w][DIAG_NSUM] = mx;
    }
    __syncthreads();
    if (threadIdx.x <= DIAG_NSUM) {
        const int k = threadIdx.x;
        double a = sh[0][k];
        for (int j = 1; j < DIAG_THREADS / 32; ++j) a = k == DIAG_NSUM ? (sh[j][k] > a ? sh[j][k] : a) : a + sh[j][k];
        partial[(long long)blockIdx.x * (DIAG_NSUM + 1) + k] = a;
    }
}

// one block: adds the block partials in index order, reads the probe sites
template <typename T>
__global__ void k_diag_final(const double* __restrict__ partial, int blocks, const T* __restrict__ m, int nx, int ny, int nz,
                             const int* __restrict__ probes, int nprobes, double* __restrict__ out /* [NSUM + 1 + nprobes] */) {
    const int k = threadIdx.x;
    if (k <= DIAG_NSUM) {
        double a = partial[k];
        for (int b = 1; b < blocks; ++b) {
            const double v = partial[(long long)b * (DIAG_NSUM + 1) + k];
            a = k == DIAG_NSUM ? (v > a ? v : a) : a + v;
        }
        out[k] = a;
    }
    for (int p = k; p < nprobes; p += blockDim.x) {
        const int x = probes[3 * p], y = probes[3 * p + 1], z = probes[3 * p + 2];
        out[DIAG_NSUM + 1 + p] = (double)m[((long long)z * ny + y) * nx + x];
    }
}

// k_diag_final for probe coordinates the host never saw (lbwp_diagnostics_static: they are device data): the same sums
// in the same order; a probe outside the box reads nothing and reports NaN; out[DIAG_NSUM - 1] (unused sum) is 0.
template <typename T>
__global__ void k_diag_final_checked(const double* __restrict__ partial, int blocks, const T* __restrict__ m, int nx, int ny, int nz,
                                     const int* __restrict__ probes, int nprobes, double* __restrict__ out /* [NSUM + 1 + nprobes] */) {
    const int k = threadIdx.x;
    if (k <= DIAG_NSUM) {
        double a = partial[k];
        for (int b = 1; b < blocks; ++b) {
            const double v = partial[(long long)b * (DIAG_NSUM + 1) + k];
            a = k == DIAG_NSUM ? (v > a ? v : a) : a + v;
        }
        out[k] = a;
    }
    for (int p = k; p < nprobes; p += blockDim.x) {
        const int x = probes[3 * p], y = probes[3 * p + 1], z = probes[3 * p + 2];
        const bool inside = x >= 0 && x < nx && y >= 0 && y < ny && z >= 0 && z < nz;
        out[DIAG_NSUM + 1 + p] = inside ? (double)m[((long long)z * ny + y) * nx + x] : __longlong_as_double(0x7ff8000000000000ll);
    }
}

}  // namespace lbwp
