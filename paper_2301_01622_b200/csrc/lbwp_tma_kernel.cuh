// lbwp_tma_kernel.cuh -- the z-marching TMA kernel and its two epilogues (see lbwp_tma.cuh).
#pragma once
#include "lbwp_tma_step.cuh"

namespace lbwp {

// BGK collision in moment space (Eq. 8) of the finished sums a = (drho, j, dP_aa = P_aa - 1/3, P_ab)
// of Eq. 1-3, written as the node's S-form scaled by the common denominator of the lattice weights (1/216, D3Q19:
// 1/36): out = c (drho - (3/2) tr S, 3 j, (9/2) S_aa, 9 S_ab), S = omega rho u u + (1 - omega)(P - rho cs^2 I).
// The ONE implementation of the collision on the TMA path: over all nodes a thread owns at once (packed
// FMUL2/FFMA2 for the fp32 pair) or, through collide_sform_node, for a single node.
template <typename T, typename V, int N, int Q>
__device__ __forceinline__ void collide_sform_v(const V (&a)[10], T omega, V (&out)[10]) {
    const T c = Q == 27 ? T(1.0 / 216.0) : T(1.0 / 36.0);
    V irho;
#pragma unroll
    for (int n = 0; n < N; ++n) irho.set(n, rcp_t<T>(T(1) + a[0].get(n)));
    const V om = V::bc(omega), om1 = V::bc(T(1) - omega);
    const V ux = a[1] * irho, uy = a[2] * irho, uz = a[3] * irho;
    const V wx = om * a[1], wy = om * a[2], wz = om * a[3];          // omega rho u
    const V iso = a[0] * V::bc(T(1.0 / 3.0));                        // rho cs^2 - 1/3
    const V sxx = vfma(wx, ux, om1 * (a[4] - iso));
    const V syy = vfma(wy, uy, om1 * (a[5] - iso));
    const V szz = vfma(wz, uz, om1 * (a[6] - iso));
    const V sxy = vfma(wx, uy, om1 * a[7]);
    const V sxz = vfma(wx, uz, om1 * a[8]);
    const V syz = vfma(wy, uz, om1 * a[9]);
    out[0] = V::bc(c) * vfma(V::bc(T(-1.5)), sxx + syy + szz, a[0]);
    const V c3 = V::bc(T(3) * c), c45 = V::bc(T(4.5) * c), c9 = V::bc(T(9) * c);
    out[1] = c3 * a[1]; out[2] = c3 * a[2]; out[3] = c3 * a[3];
    out[4] = c45 * sxx; out[5] = c45 * syy; out[6] = c45 * szz;
    out[7] = c9 * sxy; out[8] = c9 * sxz; out[9] = c9 * syz;
}
template <typename T, int Q>
__device__ __forceinline__ void collide_sform_node(const T (&a)[10], T omega, T (&out)[10]) {
    Vec<T, 1> av[10], ov[10];
#pragma unroll
    for (int f = 0; f < 10; ++f) av[f].v = a[f];
    collide_sform_v<T, Vec<T, 1>, 1, Q>(av, omega, ov);
#pragma unroll
    for (int f = 0; f < 10; ++f) out[f] = ov[f].v;
}

// stores of one node's S-form with its periodic images in the x ghost columns (reading C13; nx >= 2 here): x = -1
// and x = nx, and x = nx + 1 (read by the x-paired kernel from buffer 0)
template <typename T>
__device__ __forceinline__ void store_sform_node(const XLayout& L, T* __restrict__ dst, const T (&out)[10], int x, int y, int z) {
    const long long F = L.field;
    T* __restrict__ d = dst + xidx(L, x, y, z);
#pragma unroll
    for (int f = 0; f < 10; ++f) d[f * F] = out[f];
    if (x == 0 || x == L.nx - 1) {
        T* __restrict__ g = x == 0 ? d + L.nx : d - L.nx;
#pragma unroll
        for (int f = 0; f < 10; ++f) g[f * F] = out[f];
    }
    if (x == 1) {
#pragma unroll
        for (int f = 0; f < 10; ++f) d[f * F + L.nx] = out[f];
    }
}

// Epilogue of one finished output node.  acc = (drho, j, dP_aa = P_aa - 1/3, P_ab), Eq. 1-3.
//   EPI_SFORM:   collide (Eq. 8) and store the S-form
//   EPI_MOMENTS: store rho, u = j / rho (reading C11), P  (external dense layout)
template <typename T, int EPI, int Q = 27>
__device__ __forceinline__ void epilogue_node(const TmaStepParams<T>& p, const T (&a)[10], int x, int y, int z) {
    const XLayout& L = p.L;
    if (x == L.nx) x = 0;   // x-paired mode: the last pair of a row ends on node 0
    if (EPI == EPI_MOMENTS) {
        const T irho = rcp_t<T>(T(1) + a[0]);
        const long long n = (long long)L.nx * L.ny * L.nz;
        T* __restrict__ d = p.dst + ((long long)z * L.ny + y) * L.nx + x;
        d[0] = T(1) + a[0];
        d[n] = a[1] * irho; d[2 * n] = a[2] * irho; d[3 * n] = a[3] * irho;
        d[4 * n] = a[4] + T(1.0 / 3.0); d[5 * n] = a[5] + T(1.0 / 3.0); d[6 * n] = a[6] + T(1.0 / 3.0);
        d[7 * n] = a[7]; d[8 * n] = a[8]; d[9 * n] = a[9];
        return;
    }
    T out[10];
    collide_sform_node<T, Q>(a, p.omega, out);
    store_sform_node<T>(L, p.dst, out, x, y, z);
}

// x-paired fp32 nodes (x, x+1): one 8-byte store per field (the destination buffer's parity makes the pair aligned,
// see TmaCfg).  Ghost images: writing buffer 1 (sh = 1, x odd) the last pair of a row is (nx-1, node 0), stored at
// the columns of x = nx-1 and the ghost x = nx, and once more at the columns of the ghost x = -1 and of node 0;
// writing buffer 0 (sh = 0, x even) the pair (0, 1) is stored once more at the ghost columns x = nx, nx+1.
__device__ __forceinline__ void store_sform_pair(const XLayout& L, float* __restrict__ dst, const f32x2 (&out)[10], int x,
                                                 int y, int z) {
    const long long F = L.field;
    float* __restrict__ d = dst + xidx(L, x, y, z);
#pragma unroll
    for (int f = 0; f < 10; ++f) *reinterpret_cast<float2*>(d + f * F) = make_float2(out[f].x, out[f].y);
    if (x == 0 || x + 1 == L.nx) {
        float* __restrict__ e = x == 0 ? d + L.nx : d - L.nx;
#pragma unroll
        for (int f = 0; f < 10; ++f) *reinterpret_cast<float2*>(e + f * F) = make_float2(out[f].x, out[f].y);
    }
}
template <typename V>
__device__ __forceinline__ void store_sform_pair(const XLayout&, double*, const V (&)[10], int, int, int) {}

// Two-component runs (lbwp_tma2.cuh): the finished sums are stored as they are, (rhoA, drho, j, dP_aa,
// P_ab) plus the phase field phi = (rhoA - rhoB)/rho the next collision pass differentiates.
template <typename T>
__device__ __forceinline__ void store_raw2_node(const XLayout& L, T* __restrict__ dst, const T (&a)[11], int x, int y, int z) {
    const long long F = L.field;
    T* __restrict__ d = dst + xidx(L, x, y, z);
    d[0] = a[10];
#pragma unroll
    for (int f = 0; f < 10; ++f) d[(1 + f) * F] = a[f];
    const T rho = T(1) + a[0];
    d[11 * F] = (a[10] + a[10] - rho) * rcp_t<T>(rho);
}

// Two-component sums (drho, j, dP_aa, P_ab, rhoA) written as the external moments (rhoA, rhoB, u, P), dense [11][nz][ny][nx]
template <typename T>
__device__ __forceinline__ void store_dense2(const XLayout& L, T* __restrict__ ext, const T (&a)[11], int x, int y, int z) {
    const long long n = (long long)L.nx * L.ny * L.nz;
    T* __restrict__ d = ext + ((long long)z * L.ny + y) * L.nx + x;
    const T rho = T(1) + a[0];
    const T irho = rcp_t<T>(rho);
    d[0] = a[10];
    d[n] = rho - a[10];
    d[2 * n] = a[1] * irho; d[3 * n] = a[2] * irho; d[4 * n] = a[3] * irho;
    d[5 * n] = a[4] + T(1.0 / 3.0); d[6 * n] = a[5] + T(1.0 / 3.0); d[7 * n] = a[6] + T(1.0 / 3.0);
    d[8 * n] = a[7]; d[9 * n] = a[8]; d[10 * n] = a[9];
}

// Work decomposition: item = (z chunk, tile row, tile column), x fastest, so that items handled at
// the same time by neighbouring CTAs are spatial neighbours and their halo reads meet in L2.
struct TmaItem {
    int x0, y0, z0, nin, ym, yp;
};
template <typename C>
__device__ __forceinline__ TmaItem tma_item(const XLayout& L, int lz, int gx, int gy, int item) {
    TmaItem t;
    const int tx = item % gx, r = item / gx;
    const int ty = r % gy, tz = r / gy;
    t.x0 = tx * C::TX;
    t.y0 = ty * C::TY;
    t.z0 = tz * lz;
    t.nin = min(lz, L.nz - t.z0) + 2;                       // input planes z0-1 .. z1
    t.ym = t.y0 == 0 ? L.ny - 1 : t.y0 - 1;                 // halo rows wrap in y (reading C13)
    t.yp = t.y0 + C::TY >= L.ny ? 0 : t.y0 + C::TY;
    return t;
}

// CTA b handles items b, b + gridDim.x, ... (gridDim.x = number of items gives one item per CTA and
// leaves the order to the hardware scheduler; a smaller grid makes the CTAs persistent).  Warp
// specialisation: the last warpgroup is the TMA producer (one elected lane of its first warp; the other three
// warps only take part in the register hand-over), the first NW warps consume.  The stage ring runs straight
// across item boundaries.
// Registers: the CTA is launched with tma_max_regs() per thread; the producer warpgroup then drops to 24 and the
// consumers pick up what it released (setmaxnreg, SASS USETMAXREG): 96 -> 112 for 16 consumer warps.
constexpr int TMA_PRODUCER_THREADS = 128;
constexpr int TMA_PRODUCER_REGS = 24;
__host__ __device__ constexpr int tma_max_regs(int threads, int minb) {
    const int r = 65536 / (minb * threads) / 8 * 8;
    return r > 248 ? 248 : r;
}
__host__ __device__ constexpr int tma_consumer_regs(int consumers, int minb) {
    const int launch = tma_max_regs(consumers + TMA_PRODUCER_THREADS, minb);
    const int r = (launch + (launch - TMA_PRODUCER_REGS) * TMA_PRODUCER_THREADS / consumers) / 8 * 8;
    return r > 248 ? 248 : r;
}
template <int N> __device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

template <typename T, typename C, int EPI, int MINB>
__global__ void __maxnreg__(tma_max_regs(C::NT + TMA_PRODUCER_THREADS, MINB))
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
    const int gx = L.nx / C::TX, gy = L.ny / C::TY;
    const int nitems = gx * gy * ((L.nz + p.lz - 1) / p.lz);
    int item = blockIdx.x;
    if (item >= nitems) return;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < C::NS; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), C::NW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid >= C::NT) {
        // ---- producer warpgroup: one lane fills every free stage, up to NS planes ahead of the consumers ----
        setmaxnreg_dec<TMA_PRODUCER_REGS>();
        if (tid != C::NT) return;
        const uint64_t keep = l2_policy_evict_last();
        int ps = 0;
        uint32_t pround = 0;
        for (; item < nitems; item += gridDim.x) {
            const TmaItem t = tma_item<C>(L, p.lz, gx, gy, item);
            for (int i = 0; i < t.nin; ++i) {
                if (pround > 0) mbar_wait(empty(ps), (pround - 1u) & 1u);   // previous use released
                int z = t.z0 - 1 + i;
                z = z < 0 ? z + L.nz : (z >= L.nz ? z - L.nz : z);          // z wraps on the load side
                const uint32_t dst = base + (uint32_t)(ps * C::STAGE * sizeof(T));
                mbar_expect_tx(full(ps), C::STAGE_TX_BYTES);
                const int bx = C::PX ? t.x0 + 16 / (int)sizeof(T) : t.x0 + L.ox - C::OX;   // box start column (16-byte aligned)
                tma_load_4d(dst, &map_main, full(ps), bx, 0, t.y0, z, keep);
                tma_load_4d(dst + (uint32_t)(C::OFF_YM * sizeof(T)), &map_row, full(ps), bx, 0, t.ym, z, keep);
                tma_load_4d(dst + (uint32_t)(C::OFF_YP * sizeof(T)), &map_row, full(ps), bx, 0, t.yp, z, keep);
                if (++ps == C::NS) { ps = 0; ++pround; }
            }
        }
        return;
    }

    // ---- consumer warps ----
    setmaxnreg_inc<tma_consumer_regs(C::NT, MINB)>();
    const int tc = tid % C::COLS_T, tr = tid / C::COLS_T;
    // node n of the thread: column tx + n * DX, row tr + n * DY of the tile
    constexpr int DX = C::PX ? 1 : 0, DY = C::PX ? 0 : C::ROWS_T;
    const int tx = C::PX ? 2 * tc : tc;
    // element offsets (within a stage) of the three source rows of each owned node
    int r[C::NPT][3];
#pragma unroll
    for (int n = 0; n < C::NPT; ++n) {
        const int ty = tr + n * DY;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const int row = ty - 1 + j;
            r[n][j] = (row < 0 ? C::OFF_YM : row >= C::TY ? C::OFF_YP : row * C::ROW) + C::OX + tx + n * DX;
        }
    }

    V a0[C::NA], a1[C::NA], a2[C::NA];
#pragma unroll
    for (int f = 0; f < C::NA; ++f) a0[f] = a1[f] = a2[f] = V::bc(T(0));

    TmaItem ct = tma_item<C>(L, p.lz, gx, gy, item);
    int i = 0;            // input plane counter within the item
    int s = 0;            // stage of the current plane
    uint32_t par = 0;     // phase parity of this round of the ring

    // The first two planes of an item only prime the accumulators (their "finished" planes belong to
    // the z halo and are not stored), so nothing has to be reset at an item boundary.
    auto plane = [&](V(&P)[C::NA], V(&Cc)[C::NA], V(&N)[C::NA]) {
        int rs[C::NPT][3];
#pragma unroll
        for (int n = 0; n < C::NPT; ++n)
#pragma unroll
            for (int j = 0; j < 3; ++j) rs[n][j] = r[n][j] + s * C::STAGE;
        mbar_wait(full(s), par);
        if constexpr (C::NC == 2 && C::Q == 27) S::consume2c(sm, rs, P, Cc, N);
        else if constexpr (C::NC == 2) S::consume2c19(sm, rs, P, Cc, N);
        else if constexpr (C::Q == 27) S::consume(sm, rs, P, Cc, N);
        else S::consume19(sm, rs, P, Cc, N);
        // P[0] (all W and O brackets), Cc[0] (all E brackets, the D3Q19 corners included) and, for two components, the
        // colour sums P[10], Cc[10] (rA, K, R0) together depend on every load of the plane
        consumer_release_after(empty(s), tid, ((P[0] + Cc[0]) + (P[C::NA - 1] + Cc[C::NA - 1])).get(0), p.dep_mask);
        if (i >= 2) {                               // this input plane completes output plane z0 + i - 2
            // collision over the thread's nodes at once, except where it costs registers the stencil needs
            // (fp32 D3Q27 at 96 registers: packed epilogue spills and measured 56 vs 62 GLUPS)
            constexpr bool kVectorEpilogue = C::PX || !(C::Q == 27 && C::NPT == 2);
            if constexpr (C::NC == 2) {
#pragma unroll
                for (int n = 0; n < C::NPT; ++n) {
                    T acc[C::NA];
#pragma unroll
                    for (int f = 0; f < C::NA; ++f) acc[f] = P[f].get(n);
                    store_raw2_node<T>(L, p.dst, acc, ct.x0 + p.sh + tx + n * DX, ct.y0 + tr + n * DY, ct.z0 + i - 2);
                }
            } else if (EPI == EPI_SFORM && kVectorEpilogue) {
                V out[10];
                collide_sform_v<T, V, C::NPT, C::Q>(reinterpret_cast<const V(&)[10]>(P), p.omega, out);
                if constexpr (C::PX != 0) {
                    store_sform_pair(L, p.dst, out, ct.x0 + p.sh + tx, ct.y0 + tr, ct.z0 + i - 2);
                } else {
#pragma unroll
                    for (int n = 0; n < C::NPT; ++n) {
                        T o[10];
#pragma unroll
                        for (int f = 0; f < 10; ++f) o[f] = out[f].get(n);
                        store_sform_node<T>(L, p.dst, o, ct.x0 + p.sh + tx, ct.y0 + tr + n * DY, ct.z0 + i - 2);
                    }
                }
            } else {
#pragma unroll
                for (int n = 0; n < C::NPT; ++n) {
                    T acc[10];
#pragma unroll
                    for (int f = 0; f < 10; ++f) acc[f] = P[f].get(n);
                    epilogue_node<T, EPI, C::Q>(p, acc, ct.x0 + p.sh + tx + n * DX, ct.y0 + tr + n * DY, ct.z0 + i - 2);
                }
            }
        }
        if (++s == C::NS) { s = 0; par ^= 1u; }
        if (++i == ct.nin) {
            i = 0;
            item += gridDim.x;
            if (item < nitems) ct = tma_item<C>(L, p.lz, gx, gy, item);
        }
    };

    while (true) {   // accumulator sets rotate with period 3
        plane(a0, a1, a2);
        if (item >= nitems) break;
        plane(a1, a2, a0);
        if (item >= nitems) break;
        plane(a2, a0, a1);
        if (item >= nitems) break;
    }
}

}  // namespace lbwp
