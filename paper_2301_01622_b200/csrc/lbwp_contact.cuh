// lbwp_contact.cuh -- near-contact repulsion (Eq. 10; readings C20-C24) on the fused two-component
// TMA state (lbwp_tma2g.cuh): ONE pointwise pass after every step (and after the import), in place.
//
// The state holds every node's moments already collided (BGK, Eq. 8) in S-form, x 1/216 (D3Q19: x 1/36), plus
// rA = rhoA / rho.  The force of the collision that produced them depends on the colour field of the same time
// level, i.e. on the rA values the step kernel has just written -- of the node's neighbours too, so it cannot be
// applied in that kernel's epilogue.  This pass
//   1. differentiates phi = 2 rA - 1 at the node:  G = 3 sum_i w_i c_i phi(x + c_i) = 6 sum_i w_i c_i rA(x + c_i);
//   2. at interface nodes (|G| > G_I = 0.05) walks along the lattice direction closest to the outward normal -G/|G|
//      (first in the order cz, cy, cx on a tie) and differentiates again at each node on the way: the first interface
//      node within h_c whose gradient opposes G is a facing interface, F = (A_h / 2) G (reading C22-C23);
//   3. where F != 0, replaces the node's collided moments by the ones Guo's forcing gives (reading C24):
//      u* = u + F / (2 rho) in the quadratic term, j + F in the linear one, S += (1 - omega/2)(u* F + F u*), i.e.
//        dS_ab = omega [ (u_a F_b + F_a u_b) / 2 + F_a F_b / (4 rho) ] + (1 - omega/2)(u*_a F_b + F_a u*_b),
//        J += 3 F,  Sd_a += 4.5 dS_aa,  So_ab += 9 dS_ab,  a -= 1.5 tr dS            (all x the state's scale),
//      with rho, u = j / rho recovered from the S-form itself.
// Only rA is read at other nodes and only the fields 0..9 of the own node are written, so the pass is race-free in
// place.  Traffic: rA once per node (a CTA whose box and halo lie in one bulk phase leaves after reading them; elsewhere
// the 27 neighbours come from L1/L2) and ten fields read + written at the few nodes of a film between two interfaces:
// about 5 % of the step's.
#pragma once
#include "lbwp_tma.cuh"

namespace lbwp {

template <typename T>
struct ContactParams {
    XLayout L;              // layout of the buffer (the x-paired kernel keeps buffer 1 one column to the right)
    T* __restrict__ state;  // eleven fields
    T omega, A_h, h_c;
};

// G at node (x, y, z), 0 <= x < nx (x +- 1 from the ghost columns), y and z wrapped here (reading C13)
template <typename T, int Q>
__device__ __forceinline__ void contact_gradient(const XLayout& L, const T* __restrict__ ra, int x, int y, int z, T& gx, T& gy, T& gz) {
    const int ym = y == 0 ? L.ny - 1 : y - 1, yp = y + 1 == L.ny ? 0 : y + 1;
    const int zm = z == 0 ? L.nz - 1 : z - 1, zp = z + 1 == L.nz ? 0 : z + 1;
    gx = gy = gz = T(0);
#pragma unroll
    for (int cz = -1; cz <= 1; ++cz)
#pragma unroll
        for (int cy = -1; cy <= 1; ++cy) {
            const long long row = xidx(L, x, cy < 0 ? ym : cy > 0 ? yp : y, cz < 0 ? zm : cz > 0 ? zp : z);
#pragma unroll
            for (int cx = -1; cx <= 1; ++cx) {
                const int n2 = cx * cx + cy * cy + cz * cz;
                if (n2 == 0 || (Q == 19 && n2 == 3)) continue;
                const T w = Q == 27 ? (n2 == 1 ? T(2.0 / 27.0) : n2 == 2 ? T(1.0 / 54.0) : T(1.0 / 216.0))
                                    : (n2 == 1 ? T(1.0 / 18.0) : T(1.0 / 36.0));
                const T v = w * ra[row + cx];
                if (cx) gx += T(cx) * v;
                if (cy) gy += T(cy) * v;
                if (cz) gz += T(cz) * v;
            }
        }
    gx *= T(6); gy *= T(6); gz *= T(6);
}

// steps 1-3 at one node
template <typename T, int Q>
__device__ __forceinline__ void contact_node(const ContactParams<T>& p, int x, int y, int z) {
    const XLayout& L = p.L;
    const long long F = L.field;
    const T* __restrict__ ra = p.state + 10 * F;
    T gx, gy, gz;
    contact_gradient<T, Q>(L, ra, x, y, z, gx, gy, gz);
    const T GI2 = T(0.05 * 0.05);
    if (!(gx * gx + gy * gy + gz * gz > GI2)) return;
    int mx = 0, my = 0, mz = 0;
    T best = T(-1e30), len = T(1);
#pragma unroll
    for (int cz = -1; cz <= 1; ++cz)
#pragma unroll
        for (int cy = -1; cy <= 1; ++cy)
#pragma unroll
            for (int cx = -1; cx <= 1; ++cx) {
                const int n2 = cx * cx + cy * cy + cz * cz;
                if (n2 == 0 || (Q == 19 && n2 == 3)) continue;
                const T norm = n2 == 1 ? T(1) : n2 == 2 ? T(1.4142135623730951) : T(1.7320508075688772);
                const T inorm = n2 == 1 ? T(1) : n2 == 2 ? T(0.7071067811865476) : T(0.5773502691896258);
                const T cosv = -(T(cx) * gx + T(cy) * gy + T(cz) * gz) * inorm;   // directions that mirror each other tie exactly
                if (cosv > best) { best = cosv; mx = cx; my = cy; mz = cz; len = norm; }
            }
    bool facing = false;
    for (int k = 1; T(k) * len <= p.h_c && !facing; ++k) {
        int px = x + k * mx, py = y + k * my, pz = z + k * mz;                               // periodic (reading C13)
        while (px < 0) px += L.nx;
        while (px >= L.nx) px -= L.nx;
        while (py < 0) py += L.ny;
        while (py >= L.ny) py -= L.ny;
        while (pz < 0) pz += L.nz;
        while (pz >= L.nz) pz -= L.nz;
        T qx, qy, qz;
        contact_gradient<T, Q>(L, ra, px, py, pz, qx, qy, qz);
        facing = qx * qx + qy * qy + qz * qz > GI2 && qx * gx + qy * gy + qz * gz < T(0);
    }
    if (!facing) return;
    const T h = T(0.5) * p.A_h;
    const T fx = h * gx, fy = h * gy, fz = h * gz;
    // the node's collided moments: rho and u from the S-form (lbwp_tma2g.cuh: rho = 1 + (a + (Sd_x + Sd_y + Sd_z)/3) / c)
    const T c = Q == 27 ? T(1.0 / 216.0) : T(1.0 / 36.0), ic = Q == 27 ? T(216) : T(36);
    T* __restrict__ d = p.state + xidx(L, x, y, z);
    T s[10];
#pragma unroll
    for (int f = 0; f < 10; ++f) s[f] = d[f * F];
    const T rho = T(1) + (s[0] + (s[4] + s[5] + s[6]) * T(1.0 / 3.0)) * ic;
    const T irho = rcp_t<T>(rho);
    const T j3 = ic * T(1.0 / 3.0);
    const T ux = s[1] * j3 * irho, uy = s[2] * j3 * irho, uz = s[3] * j3 * irho;
    const T hr = T(0.5) * irho;
    const T sx = ux + hr * fx, sy = uy + hr * fy, sz = uz + hr * fz;                        // u*
    const T om = p.omega, k = T(1) - T(0.5) * p.omega, q = T(0.25) * irho;
    auto dS = [&](T ua, T ub, T sa, T sb, T fa, T fb) {
        return om * (T(0.5) * (ua * fb + fa * ub) + q * fa * fb) + k * (sa * fb + fa * sb);
    };
    const T dxx = dS(ux, ux, sx, sx, fx, fx), dyy = dS(uy, uy, sy, sy, fy, fy), dzz = dS(uz, uz, sz, sz, fz, fz);
    const T dxy = dS(ux, uy, sx, sy, fx, fy), dxz = dS(ux, uz, sx, sz, fx, fz), dyz = dS(uy, uz, sy, sz, fy, fz);
    s[0] -= c * T(1.5) * (dxx + dyy + dzz);
    s[1] += c * T(3) * fx; s[2] += c * T(3) * fy; s[3] += c * T(3) * fz;
    s[4] += c * T(4.5) * dxx; s[5] += c * T(4.5) * dyy; s[6] += c * T(4.5) * dzz;
    s[7] += c * T(9) * dxy; s[8] += c * T(9) * dxz; s[9] += c * T(9) * dyz;
#pragma unroll
    for (int f = 0; f < 10; ++f) d[f * F] = s[f];
    if (x < 3 || x >= L.nx - 2) {   // periodic images in the ghost columns (store_state2g: x = nx .. nx+2 and x = -2, -1)
        T* __restrict__ g = x < 3 ? d + L.nx : d - L.nx;
#pragma unroll
        for (int f = 0; f < 10; ++f) g[f * F] = s[f];
    }
}

// The force acts on the few nodes of a film between two interfaces; everywhere else step 2 leaves at once.  Two kernels
// keep the pass from paying 26 loads per node for that:
//   k_contact_scan   reads rA once, coalesced, and stores min and max of rA over every box of CONTACT_BX x CONTACT_BY x
//                    CONTACT_BZ nodes (range[0][box], range[1][box]; the last boxes may overhang the grid);
//   k_contact_fixup  a persistent kernel (its CTAs share the boxes out round-robin): for every box it takes min and max
//                    over the box and its 26 neighbours (which cover the box's halo of one node, periodic).  G_a = 6 (sum_{c_ia = +1} w_i rA_i - sum_{c_ia = -1}
//                    w_i rA_i) and sum_{c_ia = +1} w_i = 1/6 on both lattices, so |G_a| <= max - min and |G|^2 <=
//                    3 (max - min)^2: where max - min < 0.02 every node of the box has |G|^2 <= 1.2e-3 < G_I^2 = 2.5e-3
//                    and the box is skipped (exact: no node that gets a force is skipped).  The CTA runs steps 1-3 on
//                    the nodes of the remaining boxes.
constexpr int CONTACT_BX = 32, CONTACT_BY = 8, CONTACT_BZ = 4;
constexpr int CONTACT_CH = 32;    // boxes classified per round of a fix-up CTA

struct ContactBoxes {
    int nbx, nby, nbz;
    __host__ __device__ int count() const { return nbx * nby * nbz; }
};
inline ContactBoxes contact_boxes(const XLayout& L) {
    return {(L.nx + CONTACT_BX - 1) / CONTACT_BX, (L.ny + CONTACT_BY - 1) / CONTACT_BY, (L.nz + CONTACT_BZ - 1) / CONTACT_BZ};
}

// min and max over the lanes of a warp (to every lane).  fp32 goes through the integer warp reduction (redux.sync): the
// bit pattern of a float, with the low 31 bits flipped when negative, orders as a signed integer like the float does.
__device__ __forceinline__ int contact_ord(float f) { const int i = __float_as_int(f); return i ^ ((i >> 31) & 0x7fffffff); }
__device__ __forceinline__ float contact_unord(int i) { return __int_as_float(i ^ ((i >> 31) & 0x7fffffff)); }
__device__ __forceinline__ void contact_warp_range(float& lo, float& hi) {
    lo = contact_unord(__reduce_min_sync(0xffffffffu, contact_ord(lo)));
    hi = contact_unord(__reduce_max_sync(0xffffffffu, contact_ord(hi)));
}
__device__ __forceinline__ void contact_warp_range(double& lo, double& hi) {
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        const double a = __shfl_xor_sync(0xffffffffu, lo, o), b = __shfl_xor_sync(0xffffffffu, hi, o);
        lo = a < lo ? a : lo;
        hi = b > hi ? b : hi;
    }
}

// ZB: boxes along z per CTA (8 on large grids, 2 where that would leave fewer CTAs than the GPU holds)
template <typename T, int ZB>
__global__ void __launch_bounds__(CONTACT_BX * CONTACT_BY) k_contact_scan(const XLayout L, const ContactBoxes B, const T* __restrict__ ra,
                                                                          T* __restrict__ range) {
    constexpr int NW = CONTACT_BX * CONTACT_BY / 32;
    __shared__ T s_lo[ZB][NW], s_hi[ZB][NW];
    const int tid = threadIdx.y * CONTACT_BX + threadIdx.x;
    int x = blockIdx.x * CONTACT_BX + threadIdx.x, y = blockIdx.y * CONTACT_BY + threadIdx.y;
    x = x < L.nx ? x : L.nx - 1;                               // a repeated node changes neither min nor max
    y = y < L.ny ? y : L.ny - 1;
    const int bz0 = blockIdx.z * ZB;
#pragma unroll
    for (int k = 0; k < ZB; ++k) {
        if (bz0 + k >= B.nbz) break;
        T v[CONTACT_BZ];
#pragma unroll
        for (int j = 0; j < CONTACT_BZ; ++j) {
            int z = (bz0 + k) * CONTACT_BZ + j;
            z = z < L.nz ? z : L.nz - 1;
            v[j] = ra[xidx(L, x, y, z)];
        }
        T lo = v[0], hi = v[0];
#pragma unroll
        for (int j = 1; j < CONTACT_BZ; ++j) {
            lo = v[j] < lo ? v[j] : lo;
            hi = v[j] > hi ? v[j] : hi;
        }
        contact_warp_range(lo, hi);
        if ((tid & 31) == 0) { s_lo[k][tid >> 5] = lo; s_hi[k][tid >> 5] = hi; }
    }
    __syncthreads();
    if (tid < ZB && bz0 + tid < B.nbz) {
        T lo = s_lo[tid][0], hi = s_hi[tid][0];
#pragma unroll
        for (int w = 1; w < NW; ++w) {
            lo = s_lo[tid][w] < lo ? s_lo[tid][w] : lo;
            hi = s_hi[tid][w] > hi ? s_hi[tid][w] : hi;
        }
        const int box = ((bz0 + tid) * B.nby + blockIdx.y) * B.nbx + blockIdx.x;
        range[box] = lo;
        range[B.count() + box] = hi;
    }
}

template <typename T, int Q>
__global__ void __launch_bounds__(CONTACT_BX * CONTACT_BY, sizeof(T) == 4 ? 4 : 2) k_contact_fixup(const ContactParams<T> p, const ContactBoxes B,
                                                                           const T* __restrict__ range, const int split) {
    constexpr int NT = CONTACT_BX * CONTACT_BY, SUB = NT / CONTACT_CH;   // SUB threads share the 27 neighbours of a box
    static_assert(SUB == 8, "the reduction below runs over 8 adjacent lanes");
    __shared__ int4 s_list[CONTACT_CH];   // x0, y0, z0, z1 of the items to work on
    __shared__ int s_n;
    const XLayout& L = p.L;
    const int tid = threadIdx.y * CONTACT_BX + threadIdx.x;
    const int nbox = B.count();
    // An item is a box's planes part * BZ / split ... (split = 1, 2 or 4: on a small grid the planes of a box go to
    // different CTAs, there are not enough boxes to fill the GPU otherwise).  CTA b of G takes the items b, b + G,
    // b + 2 G, ...: the boxes of an interface are neighbours in the box grid, this spreads them over all CTAs.
    const long long nitem = (long long)nbox * split;
    for (long long first = 0; first + blockIdx.x < nitem; first += (long long)CONTACT_CH * gridDim.x) {
        if (tid == 0) s_n = 0;
        __syncthreads();
        const long long id = first + (long long)(tid / SUB) * gridDim.x + blockIdx.x;
        const int item = id < nitem ? (int)id : -1, box = item < 0 ? nbox : item / split, sub = tid % SUB;
        T lo = T(1e30), hi = T(-1e30);
        int bx = 0, by = 0, bz = 0;
        if (box < nbox) {
            bx = box % B.nbx; by = (box / B.nbx) % B.nby; bz = box / (B.nbx * B.nby);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int nb = sub + k * SUB;
                if (nb < 27) {
                    int qx = bx + nb % 3 - 1, qy = by + (nb / 3) % 3 - 1, qz = bz + nb / 9 - 1;
                    qx = qx < 0 ? B.nbx - 1 : qx == B.nbx ? 0 : qx;
                    qy = qy < 0 ? B.nby - 1 : qy == B.nby ? 0 : qy;
                    qz = qz < 0 ? B.nbz - 1 : qz == B.nbz ? 0 : qz;
                    const int q = (qz * B.nby + qy) * B.nbx + qx;
                    const T a = range[q], b = range[nbox + q];
                    lo = a < lo ? a : lo;
                    hi = b > hi ? b : hi;
                }
            }
        }
#pragma unroll
        for (int o = 1; o < SUB; o <<= 1) {
            const T a = __shfl_xor_sync(0xffffffffu, lo, o), b = __shfl_xor_sync(0xffffffffu, hi, o);
            lo = a < lo ? a : lo;
            hi = b > hi ? b : hi;
        }
        if (sub == 0 && box < nbox && !(hi - lo < T(0.02))) {
            const int z0 = bz * CONTACT_BZ + (item % split) * (CONTACT_BZ / split);
            s_list[atomicAdd(&s_n, 1)] = make_int4(bx * CONTACT_BX, by * CONTACT_BY, z0, min(z0 + CONTACT_BZ / split, L.nz));
        }
        __syncthreads();
        const int n = s_n;
        for (int k = 0; k < n; ++k) {
            const int4 it = s_list[k];
            const int x = it.x + threadIdx.x, y = it.y + threadIdx.y;
            if (x < L.nx && y < L.ny)
                for (int z = it.z; z < it.w; ++z) contact_node<T, Q>(p, x, y, z);
        }
        __syncthreads();
    }
}

}  // namespace lbwp
