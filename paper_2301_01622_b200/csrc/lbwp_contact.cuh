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
// place.  Traffic: rA once per node (its 27 neighbours come from L1/L2) and ten fields read + written at the few
// nodes of a film between two interfaces: about 5 % of the step's.
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

template <typename T, int Q>
__global__ void __launch_bounds__(256) k_contact_fixup(const ContactParams<T> p) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    const XLayout& L = p.L;
    if (x >= L.nx || y >= L.ny) return;
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
                const T cosv = -(T(cx) * gx + T(cy) * gy + T(cz) * gz) / norm;
                if (cosv > best) { best = cosv; mx = cx; my = cy; mz = cz; len = norm; }
            }
    bool facing = false;
    for (int k = 1; T(k) * len <= p.h_c && !facing; ++k) {
        int px = (x + k * mx) % L.nx, py = (y + k * my) % L.ny, pz = (z + k * mz) % L.nz;   // periodic (reading C13)
        px += px < 0 ? L.nx : 0; py += py < 0 ? L.ny : 0; pz += pz < 0 ? L.nz : 0;
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

}  // namespace lbwp
