// lbwp_tma2g.cuh -- two-component colour-gradient step (reading C6), fully fused: ONE kernel per time step that reads
// the eleven arrays of the state once and writes eleven ("22 hydro-arrays" with Flip-Flop, 163 "11
// arrays"): 2 x 11 x sizeof = 88 B per node and step in fp32, the method's own traffic.
//
// State per buffer (XLayout, 11 fields, two ghost columns on each side in x):
//   0..9  S-form of the total fluid after BGK only (Eq. 8; x 1/216, D3Q19: x 1/36), as in lbwp_tma.cuh
//   10    rA = rhoA / rho          (rho itself is 1 + (a + (Sd_x + Sd_y + Sd_z)/3) * 216, so rhoA, rhoB follow)
//
// One input plane z of a work item (tile TX x TY, z chunk) passes through three phases:
//   G  (gradient + local colour operators, once per SOURCE node of the plane, halo ring included): the phase field
//      phi = 2 rA - 1 is differentiated on the planes z-1, z, z+1 of a halo-2 rA tile
//      (G = 3 sum_i w_i c_i phi(x + c_i) = 6 sum_i w_i c_i rA), n = G/|G| (reading C8); the perturbation is folded
//      into the node's S-form in place (a -= (A/2)|G|, S += (A/9)|G| n n), and the recolouring vector
//      K = beta rhoA rhoB / rho n and the perturbation's rest population R0 = (A/3)|G| are written next to it;
//   C  (consume2c / consume2c19 of lbwp_tma_step.cuh, unchanged): pull + projection, the linear stencil over the
//      fifteen fields the G phase left in the stage, with the eleventh sum for colour A;
//   E  epilogue of the plane that just completed: BGK of the new total moments (Eq. 8), rA, eleven stores.
// This is the paper's order BGK -> perturbation -> recolouring -> streaming -> moments with the
// BGK moved into the producer's epilogue and the two colour operators applied where the data lands in shared memory.
//
// Shared memory: ring of NS main stages, each TY + 2 row slots [y0-1, y0 .. y0+TY-1, y0+TY] of pitch ROWP >= 15 BW
// (fields 0..10 arrive by TMA, one box per row; 11..14 = K, R0 from the G phase), and a ring of NS + 2 rA planes of
// TY + 4 rows (halo 2), loaded one plane AHEAD of the main ring so that plane z+1 is resident when plane z is
// differentiated.  Both rings complete on the main stage's `full` mbarrier.
#pragma once
#include "lbwp_tma_host.cuh"

namespace lbwp {

template <typename T, typename C>
struct Tma2gCfg {
    static constexpr int BW = C::BW, OX = C::OX, TX = C::TX, TY = C::TY, NS = C::NS;
    static constexpr int MT = 11;                                                   // fields that arrive by TMA
    static constexpr int ROWP = (15 * BW * (int)sizeof(T) + 127) / 128 * 128 / (int)sizeof(T);   // row slot pitch
    static constexpr int SLOTS = TY + 2;
    static constexpr int STAGE = SLOTS * ROWP;                                      // elements per main stage
    static constexpr uint32_t ROW_TX_BYTES = (uint32_t)(MT * BW * sizeof(T));
    // rA ring: box start 32 bytes left of the tile (halo 2 in x), rows of RBW elements with 2 rows = 128-byte multiple
    static constexpr int ROX = 32 / (int)sizeof(T);
    // ring column of stage column 0: both boxes start at 16-byte aligned columns of the padded row, the ring's box
    // RCO columns further left (x-paired mode: the stage box starts at x0 + 4, see TmaCfg, the ring box at x0)
    static constexpr int RCO = C::PX ? 4 : ROX - OX;
    static constexpr int RBW = (TX + 2 * ROX + 64 / (int)sizeof(T) - 1) / (64 / (int)sizeof(T)) * (64 / (int)sizeof(T));
    static constexpr int RROWS = TY + 4, RNS = NS + 2;
    static constexpr int RPLANE = RROWS * RBW;
    static constexpr uint32_t RPLANE_TX_BYTES = (uint32_t)(RPLANE * sizeof(T));
    static constexpr size_t SMEM = (size_t)(NS * STAGE + RNS * RPLANE) * sizeof(T) + 3 * NS * 8 + 64 + 128;   // + 64: plane flags of the G warps, bulk flag per stage
    static_assert((2 * RBW * sizeof(T)) % 128 == 0 && (ROWP * sizeof(T)) % 128 == 0, "TMA destinations are 128-byte aligned");
    static_assert(ROX >= 2 && OX >= 1, "halo");
    static_assert(RNS >= NS + 2, "an rA plane is overwritten only after the last plane that differentiates it was consumed");
};

template <typename T>
struct Tma2gParams {
    XLayout L;
    T* __restrict__ dst;   // EPI_SFORM: 11 state fields (XLayout); EPI_MOMENTS: dense external [11][nz][ny][nx]
    T omega, A, beta;
    int lz;
    int sh;                // x-paired mode: 1 if the CTA owns x0+1 .. x0+TX (reading buffer 0), else 0 (TmaCfg)
    uint32_t dep_mask = 0; // always 0: makes the consumers' release data-dependent (consumer_release_after)
};

// finished sums (drho, j, dP_aa, P_ab, rhoA) of one node -> the eleven state fields (BGK in moment space, Eq. 8), with
// the periodic images in the two ghost columns on each side (reading C13)
template <typename T, int Q>
__device__ __forceinline__ void store_state2g(const XLayout& L, T* __restrict__ dst, const T (&a)[11], T omega, int x, int y, int z) {
    T acc[10];
#pragma unroll
    for (int f = 0; f < 10; ++f) acc[f] = a[f];
    T out[11];
    collide_sform_node<T, Q>(acc, omega, reinterpret_cast<T(&)[10]>(out));
    out[10] = a[10] * rcp_t<T>(T(1) + a[0]);
    const long long F = L.field;
    T* __restrict__ d = dst + xidx(L, x, y, z);
#pragma unroll
    for (int f = 0; f < 11; ++f) d[f * F] = out[f];
    if (x < 3 || x >= L.nx - 2) {   // images at x = nx, nx+1, nx+2 and x = -2, -1
        T* __restrict__ g = x < 3 ? d + L.nx : d - L.nx;
#pragma unroll
        for (int f = 0; f < 11; ++f) g[f * F] = out[f];
    }
}

// ---- phase G of one unit = GN x-adjacent source nodes (fp32: a pair, all arithmetic packed; fp64: one node) ----
// st: main stage, ring planes rm / rc / rp = rA at z-1, z, z+1; row slot 0 .. TY+1, col 0 <-> x0 - 1 (col even for GN = 2)
// x-paired fp32 nodes (x, x+1): packed collision, one 8-byte store per field (the destination buffer's parity makes
// the pair aligned, see TmaCfg), then the periodic images element by element: x = nx-2, nx-1 also at x - nx; x = 0, 1, 2
// also at x + nx (reading buffer 0 the stencil reaches x = nx+2, reading buffer 1 x = -2); the pair (nx-1, nx) holds
// node 0 in its second element, whose image at x - nx is node 0's home column.
template <int Q>
__device__ __forceinline__ void store_state2g_pair(const XLayout& L, float* __restrict__ dst, const f32x2 (&a)[11], float omega,
                                                   int x, int y, int z) {
    f32x2 out[11];
    collide_sform_v<float, f32x2, 2, Q>(reinterpret_cast<const f32x2(&)[10]>(a), omega, reinterpret_cast<f32x2(&)[10]>(out));
    out[10].x = a[10].x * __frcp_rn(1.0f + a[0].x);
    out[10].y = a[10].y * __frcp_rn(1.0f + a[0].y);
    const long long F = L.field;
    float* __restrict__ d = dst + xidx(L, x, y, z);
#pragma unroll
    for (int f = 0; f < 11; ++f) *reinterpret_cast<float2*>(d + f * F) = make_float2(out[f].x, out[f].y);
    if (x < 3 || x + 1 >= L.nx - 2) {
#pragma unroll
        for (int n = 0; n < 2; ++n) {
            const int xe = x + n;
            if (xe < 3 || xe >= L.nx - 2) {
                float* __restrict__ e = d + n + (xe < 3 ? L.nx : -L.nx);
#pragma unroll
                for (int f = 0; f < 11; ++f) e[f * F] = n ? out[f].y : out[f].x;
            }
        }
    }
}
template <int Q, typename V>
__device__ __forceinline__ void store_state2g_pair(const XLayout&, double*, const V (&)[11], double, int, int, int) {}

template <typename T, typename C, typename G, int GN>
__device__ __forceinline__ void colour_unit(T* __restrict__ st, const T* __restrict__ rm, const T* __restrict__ rc,
                                            const T* __restrict__ rp, int row, int col, T A, T beta) {
    using GV = Vec<T, GN>;
    constexpr int Q = C::Q;
    const int sc = C::OX - 1 + col;                              // stage column of the unit's first node
    const int ro = (row + 1) * G::RBW + G::RCO + sc;             // ring: row 0 <-> y0 - 2
    // the three x taps of one ring row for the unit's nodes: m = f(x-1), c = f(x), p = f(x+1)
    auto taps = [&](const T* __restrict__ pl, int dy, GV& m, GV& c, GV& p) {
        const T* __restrict__ q = pl + ro + dy * G::RBW;
        if constexpr (GN == 2 && C::PX != 0) {   // ro is even: the pair itself is the aligned 8-byte load
            const float l = q[-1];
            const float2 b = *reinterpret_cast<const float2*>(q);
            const float h = q[2];
            m.x = l; m.y = b.x; c.x = b.x; c.y = b.y; p.x = b.y; p.y = h;
        } else if constexpr (GN == 2) {          // ro is odd: (x-1, x) and (x+1, x+2) are the two aligned 8-byte pairs
            const float2 a = *reinterpret_cast<const float2*>(q - 1), b = *reinterpret_cast<const float2*>(q + 1);
            m.x = a.x; m.y = a.y; c.x = a.y; c.y = b.x; p.x = b.x; p.y = b.y;
        } else {
            m.v = q[-1]; c.v = q[0]; p.v = q[1];
        }
    };
    GV gx, gy, gz;
    if constexpr (Q == 27) {
        // G = 6 sum_c w_c c rA, w_c = k(cx) k(cy) k(cz) / 216, k = (1, 4, 1): separable passes
        const GV four = GV::bc(T(4));
        GV X[3], Y[3], Z[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const T* __restrict__ pl = k == 0 ? rm : k == 1 ? rc : rp;
            GV d[3], sm_[3];
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                GV m, c, p;
                taps(pl, j - 1, m, c, p);
                d[j] = p - m;
                sm_[j] = vfma(four, c, p + m);
            }
            X[k] = vfma(four, d[1], d[2] + d[0]);
            Y[k] = sm_[2] - sm_[0];
            if (k != 1) Z[k] = vfma(four, sm_[1], sm_[2] + sm_[0]);
        }
        const GV w = GV::bc(T(6.0 / 216.0));
        gx = w * vfma(four, X[1], X[2] + X[0]);
        gy = w * vfma(four, Y[1], Y[2] + Y[0]);
        gz = w * (Z[2] - Z[0]);
    } else {
        // D3Q19: weights x 36 = 2 (axis), 1 (face diagonal): plus-shaped sums around each axis
        const GV two = GV::bc(T(2));
        GV m, c, p, m0, c0, p0;
        taps(rc, 0, m0, c0, p0);
        GV dsum = two * (p0 - m0);                       // x: 2 d(0,0) + d(+-y, 0) + d(0, +-z)
        GV ysum, zsum;
        taps(rc, 1, m, c, p);  dsum = dsum + (p - m); ysum = vfma(two, c, p + m);
        taps(rc, -1, m, c, p); dsum = dsum + (p - m); ysum = ysum - vfma(two, c, p + m);
        taps(rp, 0, m, c, p);  dsum = dsum + (p - m); zsum = vfma(two, c, p + m);
        taps(rm, 0, m, c, p);  dsum = dsum + (p - m); zsum = zsum - vfma(two, c, p + m);
        taps(rp, 1, m, c, p);  ysum = ysum + c; zsum = zsum + c;
        taps(rp, -1, m, c, p); ysum = ysum - c; zsum = zsum + c;
        taps(rm, 1, m, c, p);  ysum = ysum + c; zsum = zsum - c;
        taps(rm, -1, m, c, p); ysum = ysum - c; zsum = zsum - c;
        const GV w = GV::bc(T(6.0 / 36.0));
        gx = w * dsum; gy = w * ysum; gz = w * zsum;
    }
    const GV g2 = vfma(gx, gx, vfma(gy, gy, gz * gz));
    T* __restrict__ q = st + row * G::ROWP + sc;
    // Away from the interface (|G|^2 <= 1e-10, i.e. n = 0, for every node of the warp's units, reading C8) both colour
    // operators vanish identically: the S-form stays as it is and K = R0 = 0.  Exact, warp-uniform, the common case;
    // decided before the square root is taken.
    bool flat = true;
#pragma unroll
    for (int n = 0; n < GN; ++n) flat = flat && !(g2.get(n) > T(1e-10));
    auto ldv = [&](int f) { GV v;
        if constexpr (GN == 2 && C::PX != 0) { const float2 w = *reinterpret_cast<const float2*>(q + f * C::BW); v.x = w.x; v.y = w.y; }
        else {
#pragma unroll
            for (int n = 0; n < GN; ++n) v.set(n, q[f * C::BW + n]);
        }
        return v; };
    auto stv = [&](int f, const GV& v) {
        if constexpr (GN == 2 && C::PX != 0) *reinterpret_cast<float2*>(q + f * C::BW) = make_float2(v.get(0), v.get(1));
        else {
#pragma unroll
            for (int n = 0; n < GN; ++n) q[f * C::BW + n] = v.get(n);
        } };
    if (__all_sync(__activemask(), flat)) {
#pragma unroll
        for (int f = 11; f < 15; ++f) stv(f, GV::bc(T(0)));
        return;
    }
    GV ig;
#pragma unroll
    for (int n = 0; n < GN; ++n) ig.set(n, g2.get(n) > T(1e-10) ? rsqrt_t<T>(g2.get(n)) : T(0));   // reading C8
    const GV g = g2 * ig, nx = gx * ig, ny = gy * ig, nz = gz * ig;
    const T cw = Q == 27 ? T(1.0 / 216.0) : T(1.0 / 36.0);
    const GV sa = ldv(0), sxx = ldv(4), syy = ldv(5), szz = ldv(6), rA = ldv(10);
    const GV rho = vfma(GV::bc(T(1) / cw), vfma(GV::bc(T(1.0 / 3.0)), sxx + syy + szz, sa), GV::bc(T(1)));
    const GV Agc = GV::bc(cw * A) * g, hAg = GV::bc(T(0.5)) * Agc;   // c A |G| and half of it
    stv(0, sa - hAg);                                                  // a -= A |G| (1/3 + 1.5/9)
    const GV hx = hAg * nx, hy = hAg * ny, hz = hAg * nz;
    stv(4, vfma(hx, nx, sxx));                                         // Sd += 4.5 (A/9)|G| n n
    stv(5, vfma(hy, ny, syy));
    stv(6, vfma(hz, nz, szz));
    const GV ax = Agc * nx;
    stv(7, vfma(ax, ny, ldv(7)));                                      // So += 9 (A/9)|G| n n
    stv(8, vfma(ax, nz, ldv(8)));
    stv(9, vfma(Agc * ny, nz, ldv(9)));
    const GV kap = GV::bc(cw * beta) * (rA * (GV::bc(T(1)) - rA)) * rho;   // c beta rhoA rhoB / rho
    stv(11, kap * nx);
    stv(12, kap * ny);
    stv(13, kap * nz);
    stv(14, GV::bc(A * T(1.0 / 3.0)) * g);                              // rest population (A/3)|G|
}

// Thread roles: warps [0, NW) consume (phase C + E), the next warpgroup differentiates (phase G), the last warpgroup
// produces (one lane issues the TMA loads).  Barriers per stage: full (TMA landed) -> gdone (phase G finished) ->
// empty (phase C finished).  Registers are handed from the producer and G warpgroups to the consumers (setmaxnreg).
constexpr int TMA2G_G_THREADS = 128, TMA2G_G_REGS = 80;
__host__ __device__ constexpr int tma2g_threads(int consumers) { return consumers + TMA2G_G_THREADS + TMA_PRODUCER_THREADS; }
__host__ __device__ constexpr int tma2g_consumer_regs(int consumers) {
    const int launch = tma_max_regs(tma2g_threads(consumers), 1);
    const int r = (launch * tma2g_threads(consumers) - TMA_PRODUCER_THREADS * TMA_PRODUCER_REGS - TMA2G_G_THREADS * TMA2G_G_REGS) / consumers / 8 * 8;
    return r > 248 ? 248 : r;
}

template <typename T, typename C, int EPI>
__global__ void __maxnreg__(tma_max_regs(tma2g_threads(C::NT), 1))
k_step_tma2g(const __grid_constant__ CUtensorMap map_row, const __grid_constant__ CUtensorMap map_ra2, const __grid_constant__ CUtensorMap map_ra8,
             const Tma2gParams<T> p) {
    using G = Tma2gCfg<T, C>;
    using S = TmaStep<T, C>;
    using V = typename S::V;
    constexpr int Q = C::Q;
    constexpr int GN = sizeof(T) == 4 ? 2 : 1;
    static_assert(tma_max_regs(tma2g_threads(C::NT), 1) >= TMA2G_G_REGS, "the G warpgroup only ever releases registers");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 127u) & ~127u;
    T* const sm = reinterpret_cast<T*>(smem_raw + (base - smem_u32(smem_raw)));
    T* const ring = sm + G::NS * G::STAGE;
    const uint32_t ring_u32 = base + (uint32_t)(G::NS * G::STAGE * sizeof(T));
    const uint32_t bars = ring_u32 + (uint32_t)(G::RNS * G::RPLANE * sizeof(T));
    auto full = [&](int s) { return bars + 8u * s; };
    auto empty = [&](int s) { return bars + 8u * (G::NS + s); };
    auto gdone = [&](int s) { return bars + 8u * (2 * G::NS + s); };

    const XLayout& L = p.L;
    const int tid = threadIdx.x;
    const int gx = L.nx / C::TX, gy = L.ny / C::TY;
    const TmaItem t = tma_item<C>(L, p.lz, gx, gy, blockIdx.x);   // one item per CTA

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < G::NS; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), C::NW); mbar_init(gdone(s), TMA2G_G_THREADS / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid >= C::NT + TMA2G_G_THREADS) {
        // ---- producer warpgroup ----
        setmaxnreg_dec<TMA_PRODUCER_REGS>();
        if (tid != C::NT + TMA2G_G_THREADS) return;
        auto wrapz = [&](int z) { return z < 0 ? z + L.nz : (z >= L.nz ? z - L.nz : z); };
        auto wrapy = [&](int y) { return y < 0 ? y + L.ny : (y >= L.ny ? y - L.ny : y); };
        const int bx = C::PX ? t.x0 + 16 / (int)sizeof(T) : t.x0 + L.ox - C::OX;   // stage box start column (16-byte aligned)
        const int rbx = bx - G::RCO;
        const uint64_t keep = l2_policy_evict_last();
        // rA plane of relative index i (plane z0 - 1 + i) -> ring slot (i + 1) % RNS
        auto load_ra = [&](int i, uint32_t bar) {
            const int z = wrapz(wrapz(t.z0 - 1 + i));
            const uint32_t dst = ring_u32 + (uint32_t)(((i + 1) % G::RNS) * G::RPLANE * sizeof(T));
            tma_load_4d(dst, &map_ra2, bar, rbx, 10, wrapy(t.y0 - 2), z, keep);
            tma_load_4d(dst + (uint32_t)(2 * G::RBW * sizeof(T)), &map_ra8, bar, rbx, 10, t.y0, z, keep);
            tma_load_4d(dst + (uint32_t)((2 + C::TY) * G::RBW * sizeof(T)), &map_ra2, bar, rbx, 10, wrapy(t.y0 + C::TY), z, keep);
        };
        int ps = 0;
        uint32_t pround = 0;
        for (int i = 0; i < t.nin; ++i) {
            if (pround > 0) mbar_wait(empty(ps), (pround - 1u) & 1u);
            const int z = wrapz(t.z0 - 1 + i);
            const uint32_t dst = base + (uint32_t)(ps * G::STAGE * sizeof(T));
            mbar_expect_tx(full(ps), (uint32_t)G::SLOTS * G::ROW_TX_BYTES + (i == 0 ? 3u : 1u) * G::RPLANE_TX_BYTES);
            if (i == 0) { load_ra(-1, full(ps)); load_ra(0, full(ps)); }
            load_ra(i + 1, full(ps));
#pragma unroll 1
            for (int r = 0; r < G::SLOTS; ++r)
                tma_load_4d(dst + (uint32_t)(r * G::ROWP * sizeof(T)), &map_row, full(ps), bx, 0, wrapy(t.y0 - 1 + r), z, keep);
            if (++ps == G::NS) { ps = 0; ++pround; }
        }
        return;
    }

    if (tid >= C::NT) {
        // ---- phase G warpgroup: every source node of each plane (tile + halo ring) ----
        setmaxnreg_dec<TMA2G_G_REGS>();
        const int gt = tid - C::NT;
        constexpr int NU = (C::TX + 2) / GN, NUNITS = NU * G::SLOTS;
        static_assert((C::TX + 2) % GN == 0, "units tile the source row");
        // the units this thread handles in every plane: u = gt, gt + 128, ...; (row slot, unit in row) advance by
        // (128 / NU, 128 % NU) with a carry, no division in the plane loop
        const int row0 = gt / NU, cu0 = gt - row0 * NU;
        constexpr int DROW = TMA2G_G_THREADS / NU, DCU = TMA2G_G_THREADS % NU;
        // Plane-level shortcut (exact): if every rA the gradients of this plane's source nodes can reach -- the nodes
        // x0-2 .. x0+TX+1 of all TY+4 ring rows, in the planes z-1, z, z+1 -- lies within PHASE_DELTA of 0, or every
        // one within PHASE_DELTA of 1, then |G_a| = |6 sum_i w_i c_ia (rA_i - c)| <= 6 delta sum_i w_i |c_ia| = 2 delta
        // for every node, |G|^2 <= 12 delta^2 = 4.8e-11 < 1e-10: n = 0 everywhere (reading C8), both colour operators
        // vanish, and the plane only needs K = R0 = 0.  Each ring plane is classified once, when it arrives (three
        // rows per G warp, combined through shared memory), and the class travels with the plane.
        constexpr T PHASE_DELTA = T(2e-6);
        constexpr int FC0 = G::RCO + C::OX - 2, FNC = C::TX + 4, FROWS = G::RROWS / (TMA2G_G_THREADS / 32);
        static_assert(G::RROWS % (TMA2G_G_THREADS / 32) == 0 && FC0 >= 0 && FC0 + FNC <= G::RBW, "flag scan window");
        volatile uint32_t* const flags = reinterpret_cast<volatile uint32_t*>(smem_raw + (bars - smem_u32(smem_raw)) + 3 * G::NS * 8);
        volatile uint32_t* const kflat = flags + 8;   // per stage: 1 if the plane in it is bulk
        int nflag = 0;   // classifications done so far (parity selects the flag buffer)
        auto classify = [&](const T* __restrict__ pl) -> int {   // 0 mixed, 1 all near 0, 2 all near 1
            const int gw = gt >> 5, lane = gt & 31;
            bool z = true, o = true;
#pragma unroll
            for (int r = 0; r < FROWS; ++r)
#pragma unroll
                for (int k = 0; k < (FNC + 31) / 32; ++k) {            // independent loads: one latency, not nine
                    const int c = lane + 32 * k;
                    const T v = c < FNC ? pl[(gw * FROWS + r) * G::RBW + FC0 + c] : pl[(gw * FROWS + r) * G::RBW + FC0];
                    z = z && (fabs(v) <= PHASE_DELTA);              // NaN fails both
                    o = o && (fabs(v - T(1)) <= PHASE_DELTA);
                }
            const uint32_t mine = (__all_sync(0xffffffffu, z) ? 1u : 0u) | (__all_sync(0xffffffffu, o) ? 2u : 0u);
            volatile uint32_t* const f = flags + (nflag & 1) * 4;
            if (lane == 0) f[gw] = mine;
            asm volatile("bar.sync 1, %0;" ::"n"(TMA2G_G_THREADS) : "memory");   // the G warps only
            const uint32_t all = f[0] & f[1] & f[2] & f[3];
            ++nflag;
            return (all & 1u) ? 1 : (all & 2u) ? 2 : 0;
        };
        static_assert(TMA2G_G_THREADS == 128, "four flag words per buffer");
        int s = 0;
        uint32_t par = 0;
        int fm = 0, fc = 0, fp = 0, mixed_run = 0;
        for (int i = 0; i < t.nin; ++i) {
            mbar_wait(full(s), par);
            T* const st = sm + s * G::STAGE;
            const T* const rm = ring + ((i + 0) % G::RNS) * G::RPLANE;   // plane z - 1 (relative index i - 1)
            const T* const rc = ring + ((i + 1) % G::RNS) * G::RPLANE;   // plane z
            const T* const rp = ring + ((i + 2) % G::RNS) * G::RPLANE;   // plane z + 1
            if (i == 0) { fc = classify(rm); fp = classify(rc); }        // the first stage brings three ring planes
            // "mixed" is always a safe class (the per-unit path is exact), so inside an interface region -- four mixed
            // planes in a row -- only every fourth plane is looked at until a bulk plane turns up again: the scan sits
            // on the critical path of the plane (its class is needed the moment it arrives)
            fm = fc; fc = fp;
            if (mixed_run >= 4 && (i & 3) != 0) fp = 0;
            else fp = classify(rp);
            mixed_run = fp == 0 ? mixed_run + 1 : 0;
            // one bulk phase as far as this plane's gradients reach: the S-form stays, K = R0 = 0 are not even written
            // (the consumers are told through kflat[s] and skip those terms; published by the arrive on gdone below)
            const bool bulk = fm != 0 && fm == fc && fc == fp;
            if (gt == 0) kflat[s] = bulk ? 1u : 0u;
            if (!bulk) {
                int row = row0, cu = cu0;
#pragma unroll 1
                for (int u = gt; u < NUNITS; u += TMA2G_G_THREADS) {
                    colour_unit<T, C, G, GN>(st, rm, rc, rp, row, cu * GN, p.A, p.beta);
                    row += DROW; cu += DCU;
                    if (cu >= NU) { cu -= NU; ++row; }
                }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // these writes precede the stage's next TMA fill
            consumer_release(gdone(s), tid);
            if (++s == G::NS) { s = 0; par ^= 1u; }
        }
        return;
    }

    // ---- consumer warps: phases C and E ----
    setmaxnreg_inc<tma2g_consumer_regs(C::NT)>();
    const volatile uint32_t* const kflat = reinterpret_cast<const volatile uint32_t*>(smem_raw + (bars - smem_u32(smem_raw)) + 3 * G::NS * 8) + 8;
    const int tc = tid % C::COLS_T, tr = tid / C::COLS_T;
    // node n of the thread: column tx + n * DX, row tr + n * DY of the tile (x-paired: the pair 2 tc, 2 tc + 1)
    constexpr int DX = C::PX ? 1 : 0, DY = C::PX ? 0 : C::ROWS_T;
    const int tx = C::PX ? 2 * tc : tc;
    int r[C::NPT][3];   // element offsets (within a stage) of the three source rows of each owned node
#pragma unroll
    for (int n = 0; n < C::NPT; ++n)
#pragma unroll
        for (int j = 0; j < 3; ++j) r[n][j] = (tr + n * DY + j) * G::ROWP + C::OX + tx + n * DX;

    V a0[C::NA], a1[C::NA], a2[C::NA];
#pragma unroll
    for (int f = 0; f < C::NA; ++f) a0[f] = a1[f] = a2[f] = V::bc(T(0));

    int i = 0, s = 0;
    uint32_t par = 0;

    auto plane = [&](V(&P)[C::NA], V(&Cc)[C::NA], V(&N)[C::NA]) {
        mbar_wait(gdone(s), par);
        const bool kzero = kflat[s] != 0u;   // read before the stage is released
        // ---- phase C: pull + projection over the fifteen fields ----
        int rs[C::NPT][3];
#pragma unroll
        for (int n = 0; n < C::NPT; ++n)
#pragma unroll
            for (int j = 0; j < 3; ++j) rs[n][j] = r[n][j] + s * G::STAGE;
        if constexpr (Q == 27) S::consume2c(sm, rs, P, Cc, N, kzero);
        else S::consume2c19(sm, rs, P, Cc, N, kzero);
        consumer_release_after(empty(s), tid, ((P[0] + Cc[0]) + (P[C::NA - 1] + Cc[C::NA - 1])).get(0), p.dep_mask);   // see lbwp_tma_kernel.cuh
        // ---- phase E: this input plane completes output plane z0 + i - 2 ----
        if (i >= 2) {
            if constexpr (C::PX != 0 && EPI == EPI_SFORM) {
                store_state2g_pair<Q>(L, p.dst, P, p.omega, t.x0 + p.sh + tx, t.y0 + tr, t.z0 + i - 2);
            } else {
#pragma unroll
                for (int n = 0; n < C::NPT; ++n) {
                    T acc[C::NA];
#pragma unroll
                    for (int f = 0; f < C::NA; ++f) acc[f] = P[f].get(n);
                    int x = t.x0 + p.sh + tx + n * DX;
                    if (x == L.nx) x = 0;   // x-paired mode: the last pair of a row ends on node 0
                    if (EPI == EPI_SFORM) store_state2g<T, Q>(L, p.dst, acc, p.omega, x, t.y0 + tr + n * DY, t.z0 + i - 2);
                    else store_dense2<T>(L, p.dst, acc, x, t.y0 + tr + n * DY, t.z0 + i - 2);
                }
            }
        }
        if (++s == G::NS) { s = 0; par ^= 1u; }
        ++i;
    };

    while (true) {   // accumulator sets rotate with period 3
        plane(a0, a1, a2);
        if (i >= t.nin) break;
        plane(a1, a2, a0);
        if (i >= t.nin) break;
        plane(a2, a0, a1);
        if (i >= t.nin) break;
    }
}

// dense external moments [11][nz][ny][nx] (rhoA, rhoB, u, P) -> the eleven state fields, and a plain copy for t = 0
template <typename T, int Q>
__global__ void __launch_bounds__(256) k_tma2g_import(XLayout L, XLayout Lraw, const T* __restrict__ ext, T* __restrict__ state,
                                                      T* __restrict__ raw, T omega) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const long long F = L.field, c = xidx(Lraw, x, y, z);
    T m[11];
#pragma unroll
    for (int f = 0; f < 11; ++f) { m[f] = ext[f * n + e]; raw[f * F + c] = m[f]; }
    const double rho = (double)m[0] + (double)m[1];
    T a[11];
    a[0] = T(rho - 1.0);
    for (int k = 0; k < 3; ++k) a[1 + k] = T(rho * (double)m[2 + k]);
    for (int k = 0; k < 3; ++k) a[4 + k] = T((double)m[5 + k] - 1.0 / 3.0);
    for (int k = 0; k < 3; ++k) a[7 + k] = m[8 + k];
    a[10] = m[0];
    store_state2g<T, Q>(L, state, a, omega, x, y, z);
}

template <typename T>
__global__ void __launch_bounds__(256) k_tma2g_export_raw(XLayout L, const T* __restrict__ raw, T* __restrict__ ext) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const long long F = L.field, c = xidx(L, x, y, z);
#pragma unroll
    for (int f = 0; f < 11; ++f) ext[f * n + e] = raw[f * F + c];
}

// ---- host side ---------------------------------------------------------------------------------------
template <typename T, int Q> struct Tma2gGeom;
template <int Q> struct Tma2gGeom<float, Q> { using C = TmaCfg<float, 2, 64, 8, 4, Q, 2, 1>; };   // x-paired consumers
template <int Q> struct Tma2gGeom<double, Q> { using C = TmaCfg<double, 1, 32, 8, 4, Q, 2>; };

struct Tma2gPlanBase {
    XLayout Lb[2];   // per buffer: the x-paired fp32 kernel keeps buffer 1 one column to the right (TmaCfg)
    virtual ~Tma2gPlanBase() {}
    virtual int setup(const XLayout& L_, void* const buf[2]) = 0;
    virtual int stencil(int epi, int from, void* dst, double omega, double A, double beta, cudaStream_t stream) const = 0;
    virtual int import_state(const void* ext, void* state, void* raw, double omega, cudaStream_t stream) const = 0;
};

// tensor map over one field-major state buffer with an arbitrary box (bw, nf, rows, 1)
template <typename T>
inline int make_box_map(CUtensorMap* out, const void* buf, const XLayout& L, int nfields, int bw, int nf, int rows) {
    PFN_encodeTiled enc = get_encode_tiled();
    if (!enc) return -1;
    const cuuint64_t dims[4] = {(cuuint64_t)L.px, (cuuint64_t)nfields, (cuuint64_t)L.ny, (cuuint64_t)L.nz};
    const cuuint64_t strides[3] = {(cuuint64_t)L.field * sizeof(T), (cuuint64_t)L.px * sizeof(T), (cuuint64_t)L.plane * sizeof(T)};
    const cuuint32_t box[4] = {(cuuint32_t)bw, (cuuint32_t)nf, (cuuint32_t)rows, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = enc(out, sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4,
                           const_cast<void*>(buf), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : (int)r;
}

template <typename T, int Q>
struct Tma2gPlan final : Tma2gPlanBase {
    using C = typename Tma2gGeom<T, Q>::C;
    using G = Tma2gCfg<T, C>;
    XLayout L;
    CUtensorMap row_map[2], ra2_map[2], ra8_map[2];
    int lz = 0, gz = 0, grid = 0;

    static bool eligible(int nx, int ny) { return nx % C::TX == 0 && ny % C::TY == 0 && nx >= 4; }
    template <int EPI>
    static auto kernel() { return k_step_tma2g<T, C, EPI>; }

    int setup(const XLayout& L_, void* const buf[2]) override {
        L = L_;
        Lb[0] = Lb[1] = L;
        if (C::PX) Lb[1].ox += 1;
        for (int k = 0; k < 2; ++k) {
            int rc = make_box_map<T>(&row_map[k], buf[k], L, 11, C::BW, G::MT, 1);
            if (!rc) rc = make_box_map<T>(&ra2_map[k], buf[k], L, 11, G::RBW, 1, 2);
            if (!rc) rc = make_box_map<T>(&ra8_map[k], buf[k], L, 11, G::RBW, 1, C::TY);
            if (rc) return rc;
        }
        cudaError_t e = cudaFuncSetAttribute(kernel<EPI_SFORM>(), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(kernel<EPI_MOMENTS>(), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::SMEM);
        if (e != cudaSuccess) return (int)e;
        int dev = 0, sms = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        const long long cols = (long long)(L.nx / C::TX) * (L.ny / C::TY);
        tma_choose_chunks(L.nz, cols, sms, &lz, &gz);
        grid = (int)(cols * gz);
        return 0;
    }

    // one pass from buffer `from`: EPI_SFORM -> the eleven state fields of dst, EPI_MOMENTS -> dense moments in dst
    int stencil(int epi, int from, void* dst, double omega, double A, double beta, cudaStream_t stream) const override {
        Tma2gParams<T> p;
        p.L = Lb[from ^ 1]; p.dst = (T*)dst; p.omega = T(omega); p.A = T(A); p.beta = T(beta); p.lz = lz;   // EPI_SFORM writes the other buffer
        p.sh = (C::PX && from == 0) ? 1 : 0;
        if (epi == EPI_SFORM)
            kernel<EPI_SFORM>()<<<grid, tma2g_threads(C::NT), G::SMEM, stream>>>(row_map[from], ra2_map[from], ra8_map[from], p);
        else
            kernel<EPI_MOMENTS>()<<<grid, tma2g_threads(C::NT), G::SMEM, stream>>>(row_map[from], ra2_map[from], ra8_map[from], p);
        return (int)cudaGetLastError();
    }

    int import_state(const void* ext, void* state, void* raw, double omega, cudaStream_t stream) const override {
        const dim3 b(32, 8, 1), g((L.nx + 31) / 32, (L.ny + 7) / 8, L.nz);
        k_tma2g_import<T, Q><<<g, b, 0, stream>>>(Lb[0], Lb[1], (const T*)ext, (T*)state, (T*)raw, T(omega));
        return (int)cudaGetLastError();
    }
};

}  // namespace lbwp
