// lbwp_tma_step.cuh -- kernel body of the TMA-fed D3Q27 stencil step (see lbwp_tma.cuh).
#pragma once
#include "lbwp_tma.cuh"

namespace lbwp {

enum { EPI_SFORM = 0, EPI_MOMENTS = 1 };

template <typename T>
struct TmaStepParams {
    XLayout L;
    T* __restrict__ dst;   // EPI_SFORM: XLayout fields; EPI_MOMENTS: dense external [10][nz][ny][nx]
    T omega;               // 1/tau (reading C3)
    int lz;                // z planes per chunk
    T beta = T(0);         // recolouring strength (fused two-component mode only)
    int sh = 0;            // x-paired mode: 1 if the CTA owns x0+1 .. x0+TX (source buffer of even parity), else 0
    uint32_t dep_mask = 0; // always 0: makes the consumers' release data-dependent (consumer_release_after)
};

// Compile-time geometry of one instance.
// NC = 1: ten S-form fields in, ten out.  NC = 2 (colour gradient): fifteen fields per node in a stage (S-form with
// the perturbation folded in, rhoA/rho, the recolouring vector K, the rest-population term; written by the collide
// pass of lbwp_tma2.cuh, or in shared memory by the G phase of lbwp_tma2g.cuh), eleven moment sums per node (rhoA
// added).
// PX = 1 (fp32 pairs only): the thread's two nodes are x-adjacent (2t, 2t+1) instead of TY/2 rows apart: one
// LDS.64 + two LDS.32 bring the four values a field row contributes to both nodes (instead of six LDS.32), and
// results leave as STG.64.
template <typename T, int NPT_, int TX_, int TY_, int NS_, int Q_ = 27, int NC_ = 1, int PX_ = 0>
struct TmaCfg {
    static constexpr int NPT = NPT_, TX = TX_, TY = TY_, NS = NS_, Q = Q_, NC = NC_, PX = PX_;
    static_assert(PX_ == 0 || (NPT_ == 2 && sizeof(T) == 4), "x-paired mode: fp32, two nodes");
    static constexpr int M = NC_ == 1 ? 10 : 15;                    // fields per node in a stage
    static constexpr int NA = NC_ == 1 ? 10 : 11;                   // moment sums per node
    static_assert(Q_ == 27 || Q_ == 19, "lattice");
    // OX = shared-memory column of the first node the CTA owns (its halo columns are OX-1 and OX+TX).  The box
    // starts at a 16-byte aligned column of the padded row (TMA faults on any other start).  Scalar modes: the box
    // starts OX = 16 bytes left of the tile.
    // x-paired mode: OX = 1, so that a thread's pair sits at an (odd, even) column pair and its four sources
    // x-1 .. x+2 are two 8-byte aligned pairs: two conflict-free LDS.64 per field row.  TMA keeps the column parity
    // of the padded global row, and the 8-byte stores of the results want the pair at (even, odd) columns of the
    // destination, so the two ping-pong buffers differ in parity: buffer 0 keeps node x at column 4 + x, buffer 1
    // at column 5 + x.  Reading buffer 0 the CTA owns x0+1 .. x0+TX (TmaStepParams::sh = 1), reading buffer 1 it
    // owns x0 .. x0+TX-1 (sh = 0); in both cases the box starts at column x0 + 4.
    static constexpr int OX = PX_ ? 1 : 16 / (int)sizeof(T);
    static constexpr int BW = PX_ ? TX + 4 : TX + 2 * OX;     // box width: 16-byte multiple
    static constexpr int ROW = M * BW;                        // elements per tile row [field][BW]
    static constexpr int ROWS_T = PX_ ? TY : TY / NPT;        // thread rows
    static constexpr int COLS_T = PX_ ? TX / 2 : TX;          // thread columns
    static constexpr int NT = COLS_T * ROWS_T;
    static constexpr int NW = NT / 32;
    static constexpr int OFF_YM = TY * ROW;                   // halo row y0-1 (elements)
    static constexpr int OFF_YP = ((((TY + 1) * ROW * (int)sizeof(T)) + 127) / 128) * 128 / (int)sizeof(T);
    static constexpr int STAGE = (((OFF_YP + ROW) * (int)sizeof(T) + 127) / 128) * 128 / (int)sizeof(T);
    static constexpr uint32_t STAGE_TX_BYTES = (uint32_t)((TY + 2) * ROW * sizeof(T));
    static constexpr size_t SMEM = (size_t)NS * STAGE * sizeof(T) + 2 * NS * 8 + 128;
    static_assert((TY * ROW * sizeof(T)) % 128 == 0, "halo row must start 128-byte aligned");
    static_assert(NT % 32 == 0 && TY % NPT == 0, "tile/threads");
};

// x-pass of the separable (1,4,1) kernels over three brackets at cx = -1, 0, +1
template <typename V>
struct XRow { V r0, r1, r2; };
template <typename V>
__device__ __forceinline__ XRow<V> xpass(const V& m, const V& c, const V& p, const V& four) {
    XRow<V> r;
    r.r2 = p + m;
    r.r1 = p - m;
    r.r0 = vfma(four, c, r.r2);
    return r;
}

// In-plane moments m_pq = sum k(cx) k(cy) cx^p cy^q B(cx,cy) of one bracket family
template <typename V>
struct Mom6 { V m00, m10, m01, m20, m02, m11; };
template <typename V>
__device__ __forceinline__ Mom6<V> ypass(const XRow<V>& lo, const XRow<V>& mid, const XRow<V>& hi, const V& four) {
    Mom6<V> m;
    m.m02 = hi.r0 + lo.r0;
    m.m01 = hi.r0 - lo.r0;
    m.m00 = vfma(four, mid.r0, m.m02);
    m.m10 = vfma(four, mid.r1, hi.r1 + lo.r1);
    m.m11 = hi.r1 - lo.r1;
    m.m20 = vfma(four, mid.r2, hi.r2 + lo.r2);
    return m;
}

template <typename T, typename C>
struct TmaStep {
    using V = Vec<T, C::NPT>;
    static constexpr int BW = C::BW;

    // value of field f at (cx, row slot j) relative to the thread's nodes: source node x - c
    template <int F, int CX>
    __device__ static __forceinline__ V ld(const T* __restrict__ s, const int (&r)[C::NPT][3], int j) {
        V v;
#pragma unroll
        for (int n = 0; n < C::NPT; ++n) v.set(n, s[r[n][j] + F * BW - CX]);
        return v;
    }

    // brackets of one source row (cy = CY) at cx = -1, 0, +1: E, W = E + Szz, O.  WO = false skips the
    // z-dependent parts where the lattice has no direction (D3Q19: cz != 0 and cx cy != 0).
    template <int CY, bool WO_CORNERS>
    __device__ static __forceinline__ void brackets(const T* __restrict__ s, const int (&r)[C::NPT][3], V (&E)[3],
                                                    V (&W)[3], V (&O)[3]) {
        constexpr int J = 1 - CY;  // row slot of source y - cy: slot 0 = y-1, 1 = y, 2 = y+1
#pragma unroll
        for (int cx = -1; cx <= 1; ++cx) {
            const bool wo = WO_CORNERS || cx == 0 || CY == 0;
            V e, o, z;
            if (cx == -1) { e = ld<0, -1>(s, r, J); e = e + ld<4, -1>(s, r, J); e = e - ld<1, -1>(s, r, J);
                            if (wo) { o = ld<3, -1>(s, r, J); z = ld<6, -1>(s, r, J); o = o - ld<8, -1>(s, r, J); } }
            if (cx == 0) { e = ld<0, 0>(s, r, J);
                           if (wo) { o = ld<3, 0>(s, r, J); z = ld<6, 0>(s, r, J); } }
            if (cx == 1) { e = ld<0, 1>(s, r, J); e = e + ld<4, 1>(s, r, J); e = e + ld<1, 1>(s, r, J);
                           if (wo) { o = ld<3, 1>(s, r, J); z = ld<6, 1>(s, r, J); o = o + ld<8, 1>(s, r, J); } }
            if (CY != 0) {
                V syy, jy;
                if (cx == -1) { syy = ld<5, -1>(s, r, J); jy = ld<2, -1>(s, r, J); }
                if (cx == 0) { syy = ld<5, 0>(s, r, J); jy = ld<2, 0>(s, r, J); }
                if (cx == 1) { syy = ld<5, 1>(s, r, J); jy = ld<2, 1>(s, r, J); }
                e = e + syy;
                e = CY > 0 ? e + jy : e - jy;
                if (wo) {
                    V syz = cx == -1 ? ld<9, -1>(s, r, J) : cx == 0 ? ld<9, 0>(s, r, J) : ld<9, 1>(s, r, J);
                    o = CY > 0 ? o + syz : o - syz;
                }
                if (cx != 0) {
                    V sxy = cx == -1 ? ld<7, -1>(s, r, J) : ld<7, 1>(s, r, J);
                    e = (cx * CY > 0) ? e + sxy : e - sxy;
                }
            }
            E[cx + 1] = e;
            if (wo) { W[cx + 1] = e + z; O[cx + 1] = o; }
        }
    }

    template <int CY>
    __device__ static __forceinline__ void row(const T* __restrict__ s, const int (&r)[C::NPT][3], const V& four,
                                               XRow<V>& re, XRow<V>& rw, XRow<V>& ro) {
        V E[3], W[3], O[3];
        brackets_any<CY, true>(s, r, E, W, O);
        re = xpass<V>(E[0], E[1], E[2], four);
        rw = xpass<V>(W[0], W[1], W[2], four);
        ro = xpass<V>(O[0], O[1], O[2], four);
    }

    // ---- x-paired mode (C::PX): r[0][j] is the offset of node 2t in row slot j (an odd column); node 2t+1 follows ----
    // three packed pairs of field F in one source row: hi = sources (x-1, x) for cx = +1, mid = (x, x+1) for
    // cx = 0, lo = (x+1, x+2) for cx = -1.  hi and lo are the two aligned 8-byte loads themselves.
    template <int F>
    __device__ static __forceinline__ void ld3(const T* __restrict__ s, int r0, V& hi, V& mid, V& lo) {
        const T* __restrict__ q = s + r0 + F * BW;
        const float2 a = *reinterpret_cast<const float2*>(q - 1);
        const float2 b = *reinterpret_cast<const float2*>(q + 1);
        hi.x = a.x; hi.y = a.y;
        mid.x = a.y; mid.y = b.x;
        lo.x = b.x; lo.y = b.y;
    }
    template <int F>
    __device__ static __forceinline__ V ldm(const T* __restrict__ s, int r0) {
        const T* __restrict__ q = s + r0 + F * BW;
        V v; v.x = q[0]; v.y = q[1];
        return v;
    }

    template <int CY, bool WO_CORNERS>
    __device__ static __forceinline__ void brackets_px(const T* __restrict__ s, const int (&r)[C::NPT][3], V (&E)[3],
                                                       V (&W)[3], V (&O)[3]) {
        const int r0 = r[0][1 - CY];
        const bool wo_side = WO_CORNERS || CY == 0;     // z-dependent parts at cx = +-1
        V ah, am, al, xh, xm, xl, jh, jm, jl;
        ld3<0>(s, r0, ah, am, al);
        ld3<4>(s, r0, xh, xm, xl);                      // Sxx (cx^2)
        ld3<1>(s, r0, jh, jm, jl);                      // Jx  (cx)
        E[2] = (ah + xh) + jh;
        E[1] = am;
        E[0] = (al + xl) - jl;
        V zh, zm, zl;
        if (wo_side) {
            V oh, om, ol, sh, sm_, sl;
            ld3<3>(s, r0, oh, om, ol);                  // Jz
            ld3<6>(s, r0, zh, zm, zl);                  // Szz
            ld3<8>(s, r0, sh, sm_, sl);                 // Sxz (cx cz)
            O[2] = oh + sh; O[1] = om; O[0] = ol - sl;
        } else {
            O[1] = ldm<3>(s, r0);
            zm = ldm<6>(s, r0);
        }
        if (CY != 0) {
            V yh, ym, yl, kh, km, kl, ph, pm, pl;
            ld3<5>(s, r0, yh, ym, yl);                  // Syy (cy^2)
            ld3<2>(s, r0, kh, km, kl);                  // Jy  (cy)
            ld3<7>(s, r0, ph, pm, pl);                  // Sxy (cx cy)
            E[2] = E[2] + yh; E[1] = E[1] + ym; E[0] = E[0] + yl;
            if (CY > 0) { E[2] = (E[2] + kh) + ph; E[1] = E[1] + km; E[0] = (E[0] + kl) - pl; }
            else        { E[2] = (E[2] - kh) - ph; E[1] = E[1] - km; E[0] = (E[0] - kl) + pl; }
            if (wo_side) {
                V qh, qm, ql;
                ld3<9>(s, r0, qh, qm, ql);              // Syz (cy cz)
                if (CY > 0) { O[2] = O[2] + qh; O[1] = O[1] + qm; O[0] = O[0] + ql; }
                else        { O[2] = O[2] - qh; O[1] = O[1] - qm; O[0] = O[0] - ql; }
            } else {
                const V qm = ldm<9>(s, r0);
                O[1] = CY > 0 ? O[1] + qm : O[1] - qm;
            }
        }
        W[1] = E[1] + zm;
        if (wo_side) { W[2] = E[2] + zh; W[0] = E[0] + zl; }
    }

    template <int CY, bool WO_CORNERS>
    __device__ static __forceinline__ void brackets_any(const T* __restrict__ s, const int (&r)[C::NPT][3], V (&E)[3],
                                                        V (&W)[3], V (&O)[3]) {
        if constexpr (C::PX != 0) brackets_px<CY, WO_CORNERS>(s, r, E, W, O);
        else brackets<CY, WO_CORNERS>(s, r, E, W, O);
    }

    // scatter of one plane's in-plane moments into the three accumulator sets (total fluid): me = moments of the
    // E brackets (cz = 0, already weighted), mw/mo = moments of W and O (cz = +-1)
    __device__ static __forceinline__ void scatter27(const Mom6<V>& me, const Mom6<V>& mw, const Mom6<V>& mo, const V& four,
                                                     V (&P)[C::NA], V (&Cc)[C::NA], V (&N)[C::NA]) {
        // cz = 0 (k = 4)
        Cc[0] = vfma(four, me.m00, Cc[0]);
        Cc[1] = vfma(four, me.m10, Cc[1]);
        Cc[2] = vfma(four, me.m01, Cc[2]);
        Cc[4] = vfma(four, me.m20, Cc[4]);
        Cc[5] = vfma(four, me.m02, Cc[5]);
        Cc[7] = vfma(four, me.m11, Cc[7]);
        // cz = +1: arrives at plane z+1
        const V p00 = mw.m00 + mo.m00, p10 = mw.m10 + mo.m10, p01 = mw.m01 + mo.m01;
        N[0] = p00; N[1] = p10; N[2] = p01; N[3] = p00;
        N[4] = mw.m20 + mo.m20; N[5] = mw.m02 + mo.m02; N[6] = p00;
        N[7] = mw.m11 + mo.m11; N[8] = p10; N[9] = p01;
        // cz = -1: arrives at plane z-1
        const V n00 = mw.m00 - mo.m00, n10 = mw.m10 - mo.m10, n01 = mw.m01 - mo.m01;
        P[0] = P[0] + n00; P[1] = P[1] + n10; P[2] = P[2] + n01; P[3] = P[3] - n00;
        P[4] = P[4] + (mw.m20 - mo.m20); P[5] = P[5] + (mw.m02 - mo.m02); P[6] = P[6] + n00;
        P[7] = P[7] + (mw.m11 - mo.m11); P[8] = P[8] - n10; P[9] = P[9] - n01;
    }

    // D3Q19 (the paper's lattice): weights x 36 are 12 (rest), 2 (axis), 1 (face diagonal).
    // In-plane (cz = 0): (1,2,1) x (1,2,1) plus 8 on the centre; off-plane (cz = +-1): a plus shape,
    // 2 on the centre and 1 on the four in-plane axis neighbours.  Fields are pre-scaled by 1/36.
    __device__ static __forceinline__ void scatter19(const V (&El)[3], const V (&Wl)[3], const V (&Ol)[3], const V (&Em)[3],
                                                     const V (&Wm)[3], const V (&Om)[3], const V (&Eh)[3], const V (&Wh)[3],
                                                     const V (&Oh)[3], V (&P)[C::NA], V (&Cc)[C::NA], V (&N)[C::NA]) {
        const V two = V::bc(T(2)), eight = V::bc(T(8));
        // cz = 0: separable (1,2,1) passes over E, then the extra centre weight
        const XRow<V> xl = xpass<V>(El[0], El[1], El[2], two), xm = xpass<V>(Em[0], Em[1], Em[2], two),
                      xh = xpass<V>(Eh[0], Eh[1], Eh[2], two);
        Mom6<V> me = ypass<V>(xl, xm, xh, two);
        me.m00 = vfma(eight, Em[1], me.m00);
        Cc[0] = Cc[0] + me.m00; Cc[1] = Cc[1] + me.m10; Cc[2] = Cc[2] + me.m01;
        Cc[4] = Cc[4] + me.m20; Cc[5] = Cc[5] + me.m02; Cc[7] = Cc[7] + me.m11;
        // cz = +-1: plus-shaped moments of B = W + cz O over (0,0), (+-1,0), (0,+-1)
        const V wx = Wm[2] + Wm[0], wy = Wh[1] + Wl[1], ox = Om[2] + Om[0], oy = Oh[1] + Ol[1];
        const V w00 = vfma(two, Wm[1], wx + wy), o00 = vfma(two, Om[1], ox + oy);
        const V w10 = Wm[2] - Wm[0], o10 = Om[2] - Om[0];
        const V w01 = Wh[1] - Wl[1], o01 = Oh[1] - Ol[1];
        const V p00 = w00 + o00, p10 = w10 + o10, p01 = w01 + o01;
        N[0] = p00; N[1] = p10; N[2] = p01; N[3] = p00;
        N[4] = wx + ox; N[5] = wy + oy; N[6] = p00;
        N[7] = V::bc(T(0)); N[8] = p10; N[9] = p01;
        const V n00 = w00 - o00, n10 = w10 - o10, n01 = w01 - o01;
        P[0] = P[0] + n00; P[1] = P[1] + n10; P[2] = P[2] + n01; P[3] = P[3] - n00;
        P[4] = P[4] + (wx - ox); P[5] = P[5] + (wy - oy); P[6] = P[6] + n00;
        P[8] = P[8] - n10; P[9] = P[9] - n01;
    }

    // the three x taps of field F in row slot j, as populations see them: k[2] = source x-1 (cx = +1), k[1] = source x
    // (cx = 0), k[0] = source x+1 (cx = -1); either mode
    template <int F>
    __device__ static __forceinline__ void ld3any(const T* __restrict__ s, const int (&r)[C::NPT][3], int j, V (&k)[3]) {
        if constexpr (C::PX != 0) ld3<F>(s, r[0][j], k[2], k[1], k[0]);
        else { k[0] = ld<F, -1>(s, r, j); k[1] = ld<F, 0>(s, r, j); k[2] = ld<F, 1>(s, r, j); }
    }
    template <int F>
    __device__ static __forceinline__ V ld1any(const T* __restrict__ s, const int (&r)[C::NPT][3], int j) {
        if constexpr (C::PX != 0) return ldm<F>(s, r[0][j]);
        else return ld<F, 0>(s, r, j);
    }

    // consume one S-form input plane z: last contribution to output plane z-1 (P), middle one to
    // plane z (C), first one to plane z+1 (N, assigned).  Order: rho, jx, jy, jz, pxx, pyy, pzz, pxy, pxz, pyz
    __device__ static __forceinline__ void consume(const T* __restrict__ s, const int (&r)[C::NPT][3], V (&P)[C::NA],
                                                   V (&Cc)[C::NA], V (&N)[C::NA]) {
        const V four = V::bc(T(4));
        XRow<V> el, ew, eo, ml, mw_, mo_, hl, hw, ho;
        row<-1>(s, r, four, el, ew, eo);   // sources at y+1 (cy = -1)
        row<1>(s, r, four, hl, hw, ho);    // sources at y-1 (cy = +1)
        row<0>(s, r, four, ml, mw_, mo_);
        const Mom6<V> me = ypass<V>(el, ml, hl, four);
        const Mom6<V> mw = ypass<V>(ew, mw_, hw, four);
        const Mom6<V> mo = ypass<V>(eo, mo_, ho, four);
        scatter27(me, mw, mo, four, P, Cc, N);
    }

    __device__ static __forceinline__ void consume19(const T* __restrict__ s, const int (&r)[C::NPT][3], V (&P)[C::NA],
                                                     V (&Cc)[C::NA], V (&N)[C::NA]) {
        V El[3], Wl[3], Ol[3], Em[3], Wm[3], Om[3], Eh[3], Wh[3], Oh[3];
        brackets_any<-1, false>(s, r, El, Wl, Ol);   // sources at y+1 (cy = -1)
        brackets_any<1, false>(s, r, Eh, Wh, Oh);    // sources at y-1 (cy = +1)
        brackets_any<0, false>(s, r, Em, Wm, Om);
        scatter19(El, Wl, Ol, Em, Wm, Om, Eh, Wh, Oh, P, Cc, N);
    }

    // Two-component plane (reading C6; fields as written by k_colour_collide in lbwp_tma2.cuh):
    //   0..9  S-form of the total fluid with the perturbation folded in     (x 1/216)
    //   10    rA = rhoA / rho                                                (plain ratio)
    //   11..13 K = beta rhoA rhoB / rho * n                                  (x 1/216)
    //   14    R0 = (A/3)|G|, the extra rest population of the perturbation   (population units)
    // Total moments as in consume(); rhoA (sum 10) gathers the recoloured populations
    //   hA_c = rA (w_c + h_c) + w_c K.c/|c|      (+ rA R0 for the rest direction).
    template <int CY>
    __device__ static __forceinline__ void colour_row(const T* __restrict__ s, const int (&r)[C::NPT][3], const V (&E)[3],
                                                      const V (&W)[3], const V (&O)[3], const V& four, V& ae, V& aw, V& ao) {
        constexpr int J = 1 - CY;
        const V cc = V::bc(C::Q == 27 ? T(1.0 / 216.0) : T(1.0 / 36.0));
        V ra[3];
        ld3any<10>(s, r, J, ra);
        V AE[3], AW[3], AO[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const V rac = ra[k] * cc;
            AE[k] = vfma(ra[k], E[k], rac);
            AW[k] = vfma(ra[k], W[k], rac);
            AO[k] = ra[k] * O[k];
        }
        ae = vfma(four, AE[1], AE[2] + AE[0]);   // x-pass, zeroth moment only
        aw = vfma(four, AW[1], AW[2] + AW[0]);
        ao = vfma(four, AO[1], AO[2] + AO[0]);
    }

    // kzero: the plane's K and R0 fields are identically zero (and were not written: lbwp_tma2g.cuh, plane-level
    // shortcut); their terms are skipped, which leaves the sums bit for bit as adding the zeros would.
    __device__ static __forceinline__ void consume2c(const T* __restrict__ s, const int (&r)[C::NPT][3], V (&P)[C::NA],
                                                     V (&Cc)[C::NA], V (&N)[C::NA], bool kzero = false) {
        const V four = V::bc(T(4));
        V El[3], Wl[3], Ol[3], Em[3], Wm[3], Om[3], Eh[3], Wh[3], Oh[3];
        brackets_any<-1, true>(s, r, El, Wl, Ol);   // sources at y+1 (cy = -1)
        brackets_any<1, true>(s, r, Eh, Wh, Oh);    // sources at y-1 (cy = +1)
        brackets_any<0, true>(s, r, Em, Wm, Om);
        {   // total fluid: as in consume()
            const Mom6<V> me = ypass<V>(xpass<V>(El[0], El[1], El[2], four), xpass<V>(Em[0], Em[1], Em[2], four),
                                        xpass<V>(Eh[0], Eh[1], Eh[2], four), four);
            const Mom6<V> mw = ypass<V>(xpass<V>(Wl[0], Wl[1], Wl[2], four), xpass<V>(Wm[0], Wm[1], Wm[2], four),
                                        xpass<V>(Wh[0], Wh[1], Wh[2], four), four);
            const Mom6<V> mo = ypass<V>(xpass<V>(Ol[0], Ol[1], Ol[2], four), xpass<V>(Om[0], Om[1], Om[2], four),
                                        xpass<V>(Oh[0], Oh[1], Oh[2], four), four);
            scatter27(me, mw, mo, four, P, Cc, N);
        }
        // colour A, first part: sum_c w_c rA (1 + B_c)
        V ael, awl, aol, aem, awm, aom, aeh, awh, aoh;
        colour_row<-1>(s, r, El, Wl, Ol, four, ael, awl, aol);
        colour_row<1>(s, r, Eh, Wh, Oh, four, aeh, awh, aoh);
        colour_row<0>(s, r, Em, Wm, Om, four, aem, awm, aom);
        const V mae = vfma(four, aem, aeh + ael), maw = vfma(four, awm, awh + awl), mao = vfma(four, aom, aoh + aol);
        if (kzero) {
            Cc[10] = vfma(four, mae, Cc[10]);
            N[10] = maw + mao;
            P[10] = P[10] + (maw - mao);
            return;
        }
        // second part: sum_{c != 0} w_c K.c / |c|; weights x 216 / |c|: 16 (axis), 4/sqrt2 (face), 1/sqrt3 (corner)
        V kx0[3], kx1[3], kx2[3], ky0[3], ky2[3], kz0[3], kz1[3], kz2[3];   // K_a at row slot 0 (cy = +1), 1, 2
        ld3any<11>(s, r, 0, kx0); ld3any<11>(s, r, 1, kx1); ld3any<11>(s, r, 2, kx2);
        ld3any<12>(s, r, 0, ky0); ld3any<12>(s, r, 2, ky2);
        ld3any<13>(s, r, 0, kz0); ld3any<13>(s, r, 1, kz1); ld3any<13>(s, r, 2, kz2);
        const V kxa = kx1[2] - kx1[0];
        const V kxb = (kx0[2] - kx0[0]) + (kx2[2] - kx2[0]);
        const V kya = ky0[1] - ky2[1];
        const V kyb = (ky0[2] - ky2[2]) + (ky0[0] - ky2[0]);
        const V z0 = kz1[1];
        const V z1 = (kz1[2] + kz1[0]) + (kz0[1] + kz2[1]);
        const V z2 = (kz0[2] + kz0[0]) + (kz2[2] + kz2[0]);
        const V da = kxa + kya, db = kxb + kyb;
        const V f1 = V::bc(T(16)), f2 = V::bc(T(2.8284271247461903)), f3 = V::bc(T(0.57735026918962576));
        const V t0 = vfma(f1, da, f2 * db);                       // cz = 0
        const V tin = vfma(f2, da, f3 * db);                      // cz = +-1, in-plane part
        const V tz = vfma(f1, z0, vfma(f2, z1, f3 * z2));         // cz = +-1, c_z K_z part
        // rest population of the perturbation: to rho and (times rA) to rhoA of the node itself
        const V r0 = ld1any<14>(s, r, 1), rac = ld1any<10>(s, r, 1);
        Cc[0] = Cc[0] + r0;
        Cc[10] = vfma(four, mae, Cc[10]) + vfma(rac, r0, t0);
        N[10] = (maw + mao) + (tin + tz);
        P[10] = P[10] + ((maw - mao) + (tin - tz));
    }

    // The same for D3Q19: total moments as in consume19(); the colour sums use the D3Q19 weights x 36
    // (in-plane (1,2,1)^2 + 8 on the centre; off-plane a plus), K enters with 2 (axis) and 1/sqrt2 (face diagonal).
    __device__ static __forceinline__ void colour_products(const T* __restrict__ s, const int (&r)[C::NPT][3], int j,
                                                           const V (&E)[3], const V (&W)[3], const V (&O)[3], bool sides,
                                                           V (&AE)[3], V (&AW)[3], V (&AO)[3]) {
        const V cc = V::bc(T(1.0 / 36.0));
        V ra[3];
        ld3any<10>(s, r, j, ra);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const V rac = ra[k] * cc;
            AE[k] = vfma(ra[k], E[k], rac);
            if (k == 1 || sides) { AW[k] = vfma(ra[k], W[k], rac); AO[k] = ra[k] * O[k]; }
        }
    }

    __device__ static __forceinline__ void consume2c19(const T* __restrict__ s, const int (&r)[C::NPT][3], V (&P)[C::NA],
                                                       V (&Cc)[C::NA], V (&N)[C::NA], bool kzero = false) {
        const V two = V::bc(T(2)), eight = V::bc(T(8));
        V El[3], Wl[3], Ol[3], Em[3], Wm[3], Om[3], Eh[3], Wh[3], Oh[3];
        brackets_any<-1, false>(s, r, El, Wl, Ol);   // sources at y+1 (cy = -1)
        brackets_any<1, false>(s, r, Eh, Wh, Oh);    // sources at y-1 (cy = +1)
        brackets_any<0, false>(s, r, Em, Wm, Om);
        scatter19(El, Wl, Ol, Em, Wm, Om, Eh, Wh, Oh, P, Cc, N);   // total fluid: as in consume19()
        // colour A, first part: sum_c w_c rA (1 + B_c)
        V AEl[3], AWl[3], AOl[3], AEm[3], AWm[3], AOm[3], AEh[3], AWh[3], AOh[3];
        colour_products(s, r, 2, El, Wl, Ol, false, AEl, AWl, AOl);   // cy = -1 is row slot 2
        colour_products(s, r, 0, Eh, Wh, Oh, false, AEh, AWh, AOh);
        colour_products(s, r, 1, Em, Wm, Om, true, AEm, AWm, AOm);
        const V rl = vfma(two, AEl[1], AEl[2] + AEl[0]), rm = vfma(two, AEm[1], AEm[2] + AEm[0]),
                rh = vfma(two, AEh[1], AEh[2] + AEh[0]);
        const V mae = vfma(eight, AEm[1], vfma(two, rm, rh + rl));
        const V maw = vfma(two, AWm[1], (AWm[2] + AWm[0]) + (AWh[1] + AWl[1]));
        const V mao = vfma(two, AOm[1], (AOm[2] + AOm[0]) + (AOh[1] + AOl[1]));
        if (kzero) {
            Cc[10] = Cc[10] + mae;
            N[10] = maw + mao;
            P[10] = P[10] + (maw - mao);
            return;
        }
        // second part: sum_{c != 0} w_c K.c / |c|; weights x 36 / |c|: 2 (axis), 1/sqrt2 (face diagonal)
        V kx0[3], kx1[3], kx2[3], ky0[3], ky2[3], kz1[3];
        ld3any<11>(s, r, 0, kx0); ld3any<11>(s, r, 1, kx1); ld3any<11>(s, r, 2, kx2);
        ld3any<12>(s, r, 0, ky0); ld3any<12>(s, r, 2, ky2);
        ld3any<13>(s, r, 1, kz1);
        const V kxa = kx1[2] - kx1[0];
        const V kxb = (kx0[2] - kx0[0]) + (kx2[2] - kx2[0]);
        const V kya = ky0[1] - ky2[1];
        const V kyb = (ky0[2] - ky2[2]) + (ky0[0] - ky2[0]);
        const V z0 = kz1[1];
        const V z1 = (kz1[2] + kz1[0]) + (ld1any<13>(s, r, 0) + ld1any<13>(s, r, 2));
        const V da = kxa + kya, db = kxb + kyb;
        const V f2 = V::bc(T(0.70710678118654752));
        const V t0 = vfma(two, da, f2 * db);     // cz = 0: axis and in-plane face diagonals
        const V tin = f2 * da;                   // cz = +-1: (+-1, 0, cz), (0, +-1, cz)
        const V tz = vfma(two, z0, f2 * z1);     // cz = +-1: c_z K_z of (0,0,cz) and the four above
        const V r0 = ld1any<14>(s, r, 1), rac = ld1any<10>(s, r, 1);
        Cc[0] = Cc[0] + r0;
        Cc[10] = (Cc[10] + mae) + vfma(rac, r0, t0);
        N[10] = (maw + mao) + (tin + tz);
        P[10] = P[10] + ((maw - mao) + (tin - tz));
    }
};

}  // namespace lbwp
