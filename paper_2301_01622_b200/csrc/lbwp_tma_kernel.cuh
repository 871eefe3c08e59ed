// lbwp_tma_kernel.cuh -- the z-marching TMA kernel and its two epilogues (see lbwp_tma.cuh).
#pragma once
#include "lbwp_tma_step.cuh"

namespace lbwp {

// Epilogue of one finished output node.  acc = (drho, j, dP_aa = P_aa - 1/3, P_ab), Eq. 1-3.
//   EPI_SFORM:   BGK collision in moment space (Eq. 8), store the S-form scaled by 1/216
//   EPI_MOMENTS: store rho, u = j / rho (reading C11), P  (external dense layout)
template <typename T, int EPI>
__device__ __forceinline__ void epilogue_node(const TmaStepParams<T>& p, const T (&a)[10], int x, int y, int z) {
    const XLayout& L = p.L;
    const T rho = T(1) + a[0];
    const T irho = rcp_t<T>(rho);
    const T ux = a[1] * irho, uy = a[2] * irho, uz = a[3] * irho;
    if (EPI == EPI_MOMENTS) {
        const long long n = (long long)L.nx * L.ny * L.nz;
        T* __restrict__ d = p.dst + ((long long)z * L.ny + y) * L.nx + x;
        d[0] = rho;
        d[n] = ux; d[2 * n] = uy; d[3 * n] = uz;
        d[4 * n] = a[4] + T(1.0 / 3.0); d[5 * n] = a[5] + T(1.0 / 3.0); d[6 * n] = a[6] + T(1.0 / 3.0);
        d[7 * n] = a[7]; d[8 * n] = a[8]; d[9 * n] = a[9];
        return;
    }
    const T c = T(1.0 / 216.0);
    const T om1 = T(1) - p.omega;
    const T wx = p.omega * a[1], wy = p.omega * a[2], wz = p.omega * a[3];   // omega rho u
    const T iso = a[0] * T(1.0 / 3.0);                                        // rho cs^2 - 1/3
    const T sxx = fma(wx, ux, om1 * (a[4] - iso));
    const T syy = fma(wy, uy, om1 * (a[5] - iso));
    const T szz = fma(wz, uz, om1 * (a[6] - iso));
    const T sxy = fma(wx, uy, om1 * a[7]);
    const T sxz = fma(wx, uz, om1 * a[8]);
    const T syz = fma(wy, uz, om1 * a[9]);
    T out[10];
    out[0] = c * fma(T(-1.5), sxx + syy + szz, a[0]);
    out[1] = (T(3) * c) * a[1];
    out[2] = (T(3) * c) * a[2];
    out[3] = (T(3) * c) * a[3];
    out[4] = (T(4.5) * c) * sxx;
    out[5] = (T(4.5) * c) * syy;
    out[6] = (T(4.5) * c) * szz;
    out[7] = (T(9) * c) * sxy;
    out[8] = (T(9) * c) * sxz;
    out[9] = (T(9) * c) * syz;
    const long long F = L.field;
    T* __restrict__ d = p.dst + xidx(L, x, y, z);
#pragma unroll
    for (int f = 0; f < 10; ++f) d[f * F] = out[f];
    if (x == 0 || x == L.nx - 1) {   // periodic image in the x ghost column (reading C13); nx >= 2 here
        T* __restrict__ g = x == 0 ? d + L.nx : d - L.nx;
#pragma unroll
        for (int f = 0; f < 10; ++f) g[f * F] = out[f];
    }
}

template <typename T, typename C, int EPI, int MINB>
__global__ void __launch_bounds__(C::NT, MINB)
k_step_tma27(const __grid_constant__ CUtensorMap map_main, const __grid_constant__ CUtensorMap map_row,
             const TmaStepParams<T> p) {
    using S = TmaStep<T, C>;
    using V = typename S::V;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // 128-byte aligned stage ring, then the barriers
    const uint32_t base = (smem_u32(smem_raw) + 127u) & ~127u;
    T* const sm = reinterpret_cast<T*>(smem_raw + (base - smem_u32(smem_raw)));
    const uint32_t bars = base + (uint32_t)(C::NS * C::STAGE * sizeof(T));
    auto full = [&](int s) { return bars + 8u * s; };
    auto empty = [&](int s) { return bars + 8u * (C::NS + s); };

    const XLayout& L = p.L;
    const int tid = threadIdx.x;
    const int tx = tid % C::TX, tr = tid / C::TX;
    const int x0 = blockIdx.x * C::TX, y0 = blockIdx.y * C::TY;
    const int z0 = blockIdx.z * p.lz;
    const int z1 = min(z0 + p.lz, L.nz);
    const int nin = z1 - z0 + 2;                 // input planes z0-1 .. z1
    const int ym = y0 == 0 ? L.ny - 1 : y0 - 1;   // halo rows wrap in y (reading C13)
    const int yp = y0 + C::TY >= L.ny ? 0 : y0 + C::TY;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < C::NS; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), C::NW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    auto issue = [&](int i, int s) {   // input plane index i -> stage s (thread 0 only)
        int z = z0 - 1 + i;
        z = z < 0 ? z + L.nz : (z >= L.nz ? z - L.nz : z);
        const uint32_t dst = base + (uint32_t)(s * C::STAGE * sizeof(T));
        mbar_expect_tx(full(s), C::STAGE_TX_BYTES);
        tma_load_4d(dst, &map_main, full(s), x0, 0, y0, z);
        tma_load_4d(dst + (uint32_t)(C::OFF_YM * sizeof(T)), &map_row, full(s), x0, 0, ym, z);
        tma_load_4d(dst + (uint32_t)(C::OFF_YP * sizeof(T)), &map_row, full(s), x0, 0, yp, z);
    };
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < C::NS - 1; ++i)
            if (i < nin) issue(i, i);
    }

    // element offsets (within a stage) of the three source rows of each owned node, at x = tx
    int r[C::NPT][3];
#pragma unroll
    for (int n = 0; n < C::NPT; ++n) {
        const int ty = tr + n * C::ROWS_T;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const int row = ty - 1 + j;
            r[n][j] = (row < 0 ? C::OFF_YM : row >= C::TY ? C::OFF_YP : row * C::ROW) + C::OX + tx;
        }
    }

    V a0[10], a1[10], a2[10];
#pragma unroll
    for (int f = 0; f < 10; ++f) a0[f] = a1[f] = a2[f] = V::bc(T(0));

    const int x = x0 + tx;
    int i = 0;   // input plane counter

    auto plane = [&](V(&P)[10], V(&Cc)[10], V(&N)[10], int s, uint32_t par) {
        if (tid == 0) {
            const int j = i + C::NS - 1;            // refill the stage freed one plane ago
            if (j < nin) {
                const int sj = (s + C::NS - 1) % C::NS;
                if (j >= C::NS) mbar_wait(empty(sj), ((uint32_t)(j / C::NS) - 1u) & 1u);
                issue(j, sj);
            }
        }
        mbar_wait(full(s), par);
        S::consume(sm + s * C::STAGE, r, P, Cc, N);
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(empty(s));
        const int zo = z0 + i - 2;                  // plane completed by this input plane
        if (zo >= z0) {
#pragma unroll
            for (int n = 0; n < C::NPT; ++n) {
                T acc[10];
#pragma unroll
                for (int f = 0; f < 10; ++f) acc[f] = P[f].get(n);
                epilogue_node<T, EPI>(p, acc, x, y0 + tr + n * C::ROWS_T, zo);
            }
        }
        ++i;
    };

    static_assert(C::NS == 3, "stage ring and accumulator rotation share the period 3");
    uint32_t par = 0;
    while (true) {
        plane(a0, a1, a2, 0, par);
        if (i >= nin) break;
        plane(a1, a2, a0, 1, par);
        if (i >= nin) break;
        plane(a2, a0, a1, 2, par);
        if (i >= nin) break;
        par ^= 1u;
    }
}

}  // namespace lbwp
