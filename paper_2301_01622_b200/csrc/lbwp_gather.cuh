// lbwp_gather.cuh -- "gather" kernels: one thread per lattice node, Q-neighbour pull
// through L1/L2.  Generic over lattice (19|27), precision and component count; the
// fallback for every combination and the stepping stone the tiled kernel is checked
// against.  Arithmetic follows PAPER.md:77-91 in the algebraically equivalent
// "S-form":
//   post-collision population at a node with moments (rho,u,P) (Eq. 8):
//     h'_c = w_c [ rho + 3 c.j + Q_c : S ],  j = rho u,
//     S = omega rho u u + (1-omega)(P - rho cs^2 I),  Q_c = (c c - cs^2 I)/(2 cs^4)
//         = w_c [ 1 + B_c ],   B_c = da + c.J + sum_a c_a^2 Sd_a + sum_{a<b} c_a c_b So_ab
//     da = drho - 1.5 tr S, J = 3 j, Sd_a = 4.5 S_aa, So_ab = 9 S_ab.
//   The constant 1 streams to rho = 1, P_aa = 1/3 exactly, so only w_c B_c is summed
//   (deviation storage, lbwp_common.cuh).
#pragma once
#include "lbwp_common.cuh"

namespace lbwp {

// Collided node in S-form: everything a direction needs, from the stored moments.
template <typename T>
struct SNode {
    T da, Jx, Jy, Jz, Sxx, Syy, Szz, Sxy, Sxz, Syz;
};

// BGK collision in moment space (Eq. 8 before the direction-dependent contraction).
template <typename T>
__device__ __forceinline__ SNode<T> collide_sform(T drho, T ux, T uy, T uz, T dPxx, T dPyy, T dPzz, T Pxy,
                                                  T Pxz, T Pyz, T omega) {
    const T rho = T(1) + drho;
    const T om1 = T(1) - omega;
    const T orho = omega * rho;
    const T third = T(1.0 / 3.0);
    const T iso = drho * third;  // (rho cs^2 - 1/3)
    SNode<T> s;
    const T sxx = orho * ux * ux + om1 * (dPxx - iso);
    const T syy = orho * uy * uy + om1 * (dPyy - iso);
    const T szz = orho * uz * uz + om1 * (dPzz - iso);
    s.Sxy = T(9) * (orho * ux * uy + om1 * Pxy);
    s.Sxz = T(9) * (orho * ux * uz + om1 * Pxz);
    s.Syz = T(9) * (orho * uy * uz + om1 * Pyz);
    s.da = drho - T(1.5) * (sxx + syy + szz);
    s.Sxx = T(4.5) * sxx;
    s.Syy = T(4.5) * syy;
    s.Szz = T(4.5) * szz;
    const T r3 = T(3) * rho;
    s.Jx = r3 * ux;
    s.Jy = r3 * uy;
    s.Jz = r3 * uz;
    return s;
}

template <typename T, int CX, int CY, int CZ>
__device__ __forceinline__ T bracket(const SNode<T>& s) {
    T b = s.da;
    if (CX) b += T(CX) * s.Jx + s.Sxx;
    if (CY) b += T(CY) * s.Jy + s.Syy;
    if (CZ) b += T(CZ) * s.Jz + s.Szz;
    if (CX * CY) b += T(CX * CY) * s.Sxy;
    if (CX * CZ) b += T(CX * CZ) * s.Sxz;
    if (CY * CZ) b += T(CY * CZ) * s.Syz;
    return b;
}

template <typename T>
struct Acc {
    T rho, jx, jy, jz, pxx, pyy, pzz, pxy, pxz, pyz, rhoA;
};

// One direction of the pull: read the moments at y = x - c, collide there (Eq. 8),
// add the arriving population to the node's moment sums (Eq. 9, Eq. 1-3).
// NF = 1: with the near-contact body force F(y) (reading C24, Guo forcing on the reconstructed populations):
//   u* = u + F/(2 rho) in the quadratic terms, j + F in the linear term, S += (1 - omega/2)(u* F + F u*).
template <typename T, int Q, int NC, int CX, int CY, int CZ, int NF = 0>
__device__ __forceinline__ void pull_dir(const StepParams<T>& p, long long xc, Acc<T>& a) {
    constexpr int N2 = CX * CX + CY * CY + CZ * CZ;
    if (Q == 19 && N2 == 3) return;
    const T w = T(lattice_w<Q>(N2));
    const long long F = p.L.field;
    const long long y = xc - ((long long)CZ * p.L.plane + (long long)CY * p.L.px + CX);
    const T* __restrict__ s = p.src;
    T h;  // deviation of the arriving population from w_c
    if (NC == 1) {
        SNode<T> n = collide_sform<T>(s[y], s[F + y], s[2 * F + y], s[3 * F + y], s[4 * F + y], s[5 * F + y],
                                      s[6 * F + y], s[7 * F + y], s[8 * F + y], s[9 * F + y], p.omega);
        h = w * bracket<T, CX, CY, CZ>(n);
    } else {
        // colour gradient (reading C6): perturbation folded into (da, S), rest-population
        // term E0, then recolouring of the arriving population.
        const T rhoA = s[y], drho = s[F + y];
        T ux = s[2 * F + y], uy = s[3 * F + y], uz = s[4 * F + y];
        T fx = T(0), fy = T(0), fz = T(0);
        if (NF) {
            fx = p.force[y]; fy = p.force[F + y]; fz = p.force[2 * F + y];
            const T hr = T(0.5) / (T(1) + drho);
            ux += hr * fx; uy += hr * fy; uz += hr * fz;          // u*
        }
        SNode<T> n = collide_sform<T>(drho, ux, uy, uz, s[5 * F + y], s[6 * F + y],
                                      s[7 * F + y], s[8 * F + y], s[9 * F + y], s[10 * F + y], p.omega);
        if (NF) {
            // J = 3 (j + F) (collide_sform gave 3 rho u* = 3 (j + F/2)); S-form of (1 - omega/2)(u* F + F u*)
            n.Jx += T(1.5) * fx; n.Jy += T(1.5) * fy; n.Jz += T(1.5) * fz;
            const T k = T(1) - T(0.5) * p.omega;
            const T dxx = T(2) * k * ux * fx, dyy = T(2) * k * uy * fy, dzz = T(2) * k * uz * fz;
            n.da -= T(1.5) * (dxx + dyy + dzz);
            n.Sxx += T(4.5) * dxx; n.Syy += T(4.5) * dyy; n.Szz += T(4.5) * dzz;
            n.Sxy += T(9) * k * (ux * fy + uy * fx);
            n.Sxz += T(9) * k * (ux * fz + uz * fx);
            n.Syz += T(9) * k * (uy * fz + uz * fy);
        }
        const T Gx = p.grad[y], Gy = p.grad[F + y], Gz = p.grad[2 * F + y];
        const T g2 = Gx * Gx + Gy * Gy + Gz * Gz;
        const T ig = g2 > T(1e-10) ? rsqrt_t<T>(g2) : T(0);  // reading C8: |G| <= 1e-5 -> n = 0
        const T g = g2 * ig;
        const T nx = Gx * ig, ny = Gy * ig, nz = Gz * ig;
        const T Ag = p.A * g;
        // S_tot = S + (A/9)|G| n n ; drho' = drho - (A/3)|G| ; da = drho' - 1.5 tr S_tot
        n.da -= Ag * T(1.0 / 3.0) + Ag * T(1.5 / 9.0);
        n.Sxx += T(0.5) * Ag * nx * nx;
        n.Syy += T(0.5) * Ag * ny * ny;
        n.Szz += T(0.5) * Ag * nz * nz;
        n.Sxy += Ag * nx * ny;
        n.Sxz += Ag * nx * nz;
        n.Syz += Ag * ny * nz;
        h = w * bracket<T, CX, CY, CZ>(n);
        if (N2 == 0) h += Ag * T(1.0 / 3.0);
        const T rho = T(1) + drho;
        const T irho = T(1) / rho;
        const T rA = rhoA * irho;
        T hA = rA * (w + h);
        if (N2 != 0) {
            const T kappa = p.beta * rA * (rho - rhoA);  // beta rhoA rhoB / rho
            const T cn = T(CX) * nx + T(CY) * ny + T(CZ) * nz;
            const T inorm = N2 == 1 ? T(1) : N2 == 2 ? T(0.70710678118654752440) : T(0.57735026918962576451);
            hA += kappa * w * inorm * cn;
        }
        a.rhoA += hA;
    }
    a.rho += h;
    if (CX) a.jx += T(CX) * h;
    if (CY) a.jy += T(CY) * h;
    if (CZ) a.jz += T(CZ) * h;
    if (CX) a.pxx += h;
    if (CY) a.pyy += h;
    if (CZ) a.pzz += h;
    if (CX * CY) a.pxy += T(CX * CY) * h;
    if (CX * CZ) a.pxz += T(CX * CZ) * h;
    if (CY * CZ) a.pyz += T(CY * CZ) * h;
}

template <typename T, int Q, int NC, int NF = 0>
__global__ void __launch_bounds__(256) k_step_gather(const StepParams<T> p) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= p.L.nx || y >= p.L.ny) return;
    const long long xc = lidx(p.L, x, y, z);
    Acc<T> a = {};
#define LBWP_DIR(CX, CY, CZ) pull_dir<T, Q, NC, CX, CY, CZ, NF>(p, xc, a);
#define LBWP_ROW(CY, CZ) LBWP_DIR(-1, CY, CZ) LBWP_DIR(0, CY, CZ) LBWP_DIR(1, CY, CZ)
#define LBWP_PLANE(CZ) LBWP_ROW(-1, CZ) LBWP_ROW(0, CZ) LBWP_ROW(1, CZ)
    LBWP_PLANE(-1) LBWP_PLANE(0) LBWP_PLANE(1)
#undef LBWP_PLANE
#undef LBWP_ROW
#undef LBWP_DIR
    const long long F = p.L.field;
    const T irho = T(1) / (T(1) + a.rho);  // u = j / rho (Eq. 2, reading C11)
    T* __restrict__ d = p.dst;
    int k = 0;
    if (NC == 2) store_images(d + (k++) * F, p.L, x, y, z, a.rhoA);
    store_images(d + (k++) * F, p.L, x, y, z, a.rho);
    store_images(d + (k++) * F, p.L, x, y, z, a.jx * irho);
    store_images(d + (k++) * F, p.L, x, y, z, a.jy * irho);
    store_images(d + (k++) * F, p.L, x, y, z, a.jz * irho);
    store_images(d + (k++) * F, p.L, x, y, z, a.pxx);
    store_images(d + (k++) * F, p.L, x, y, z, a.pyy);
    store_images(d + (k++) * F, p.L, x, y, z, a.pzz);
    store_images(d + (k++) * F, p.L, x, y, z, a.pxy);
    store_images(d + (k++) * F, p.L, x, y, z, a.pxz);
    store_images(d + (k++) * F, p.L, x, y, z, a.pyz);
}

// Colour gradient G(y) = (1/cs^2) sum_i w_i c_i phi(y + c_i), phi = (rhoA-rhoB)/(rhoA+rhoB)
// (reading C6), from the stored (post-stream) densities.
// dst3: three fields Gx,Gy,Gz in the state layout, ghosts included.
template <typename T, int Q>
__global__ void __launch_bounds__(256) k_colour_gradient(const StepParams<T> p, T* __restrict__ dst3) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= p.L.nx || y >= p.L.ny) return;
    const long long xc = lidx(p.L, x, y, z);
    const long long F = p.L.field;
    T gx = 0, gy = 0, gz = 0;
#pragma unroll
    for (int cz = -1; cz <= 1; ++cz)
#pragma unroll
        for (int cy = -1; cy <= 1; ++cy)
#pragma unroll
            for (int cx = -1; cx <= 1; ++cx) {
                const int n2 = cx * cx + cy * cy + cz * cz;
                if (n2 == 0 || (Q == 19 && n2 == 3)) continue;
                const long long y_ = xc + ((long long)cz * p.L.plane + (long long)cy * p.L.px + cx);
                const T rhoA = p.src[y_], rho = T(1) + p.src[F + y_];
                const T phi = (rhoA + rhoA - rho) / rho;
                const T w = T(3.0 * lattice_w<Q>(n2));
                if (cx) gx += T(cx) * w * phi;
                if (cy) gy += T(cy) * w * phi;
                if (cz) gz += T(cz) * w * phi;
            }
    store_images(dst3, p.L, x, y, z, gx);
    store_images(dst3 + F, p.L, x, y, z, gy);
    store_images(dst3 + 2 * F, p.L, x, y, z, gz);
}

// Near-contact repulsion F_rep = -A_h[h(x)] n delta_I (Eq. 10; readings C20-C23): at interface nodes
// (|G| > G_I = 0.05) walk along the lattice direction closest to the outward normal -G/|G| (first in the order cz, cy,
// cx on a tie); the first interface node within h_c whose gradient opposes G is a facing interface: F = (A_h/2) G.
// grad3: Gx, Gy, Gz (ghost-padded); dst3: Fx, Fy, Fz with ghost images.
template <typename T, int Q>
__global__ void __launch_bounds__(256) k_near_contact(const StepParams<T> p, const T* __restrict__ grad3, T* __restrict__ dst3) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    const Layout& L = p.L;
    if (x >= L.nx || y >= L.ny) return;
    const long long xc = lidx(L, x, y, z);
    const long long F = L.field;
    const T gx = grad3[xc], gy = grad3[F + xc], gz = grad3[2 * F + xc];
    T fx = T(0), fy = T(0), fz = T(0);
    const T GI2 = T(0.05 * 0.05);
    if (gx * gx + gy * gy + gz * gz > GI2) {
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
        for (int k = 1; T(k) * len <= p.h_c; ++k) {
            int px = (x + k * mx) % L.nx, py = (y + k * my) % L.ny, pz = (z + k * mz) % L.nz;   // periodic (reading C13)
            px += px < 0 ? L.nx : 0; py += py < 0 ? L.ny : 0; pz += pz < 0 ? L.nz : 0;
            const long long pc = lidx(L, px, py, pz);
            const T qx = grad3[pc], qy = grad3[F + pc], qz = grad3[2 * F + pc];
            if (qx * qx + qy * qy + qz * qz > GI2 && qx * gx + qy * gy + qz * gz < T(0)) {
                const T h = T(0.5) * p.A_h;
                fx = h * gx; fy = h * gy; fz = h * gz;
                break;
            }
        }
    }
    store_images(dst3, L, x, y, z, fx);
    store_images(dst3 + F, L, x, y, z, fy);
    store_images(dst3 + 2 * F, L, x, y, z, fz);
}

}  // namespace lbwp
