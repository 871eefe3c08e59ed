// lbwp_pop.cuh -- COMPARISON POINT ONLY: standard LB "with populations"
// (PAPER.md:29, 75, 163): two-lattice pull BGK on stored populations, second-order
// equilibrium (Eq. 5).  Written in the same style as the moments kernels so the
// MLUPS / bytes-per-node comparison of PAPER.md:163 can be repeated on B200.
//
// Stored per node and direction: the POST-collision population minus w_i, in the
// same ghost-padded layout (Q fields per component).  Invariant kept by the host
// side: buf[cur] = F_t (post-collision of time t) and buf[cur^1] = F_{t-1}, whose
// pull-stream is f(t), the pre-collision populations whose Eq. 1-3 moments
// lbwp_moments returns.  At t = 0, buf[cur^1] holds the Eq. 4 populations shifted
// one link backwards so that the same pull yields them.
#pragma once
#include "lbwp_common.cuh"
#include "lbwp_gather.cuh"

namespace lbwp {

template <int Q>
__host__ __device__ constexpr int dir_index(int cx, int cy, int cz) {
    int n = 0;
    for (int z = -1; z <= 1; ++z)
        for (int y = -1; y <= 1; ++y)
            for (int x = -1; x <= 1; ++x) {
                if (Q == 19 && x * x + y * y + z * z == 3) continue;
                if (x == cx && y == cy && z == cz) return n;
                ++n;
            }
    return -1;
}

template <typename T, int Q, int CX, int CY, int CZ>
__device__ __forceinline__ void pop_pull(const Layout& L, const T* __restrict__ src, long long xc, T* f, Acc<T>& a) {
    constexpr int N2 = CX * CX + CY * CY + CZ * CZ;
    if (Q == 19 && N2 == 3) return;
    constexpr int I = dir_index<Q>(CX, CY, CZ);
    const T h = src[(long long)I * L.field + xc - ((long long)CZ * L.plane + (long long)CY * L.px + CX)];
    f[I] = h;
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

template <typename T, int Q, int CX, int CY, int CZ>
__device__ __forceinline__ void pop_collide_store(const Layout& L, T* __restrict__ dst, int x, int y, int z,
                                                  const T* f, const SNode<T>& eq, T omega) {
    constexpr int N2 = CX * CX + CY * CY + CZ * CZ;
    if (Q == 19 && N2 == 3) return;
    constexpr int I = dir_index<Q>(CX, CY, CZ);
    const T feq = T(lattice_w<Q>(N2)) * bracket<T, CX, CY, CZ>(eq);  // Eq. 5 minus w_i
    store_images(dst + (long long)I * L.field, L, x, y, z, f[I] - omega * (f[I] - feq));
}

#define LBWP_ALL_DIRS(M)                                                                            \
    M(-1, -1, -1) M(0, -1, -1) M(1, -1, -1) M(-1, 0, -1) M(0, 0, -1) M(1, 0, -1) M(-1, 1, -1)        \
    M(0, 1, -1) M(1, 1, -1) M(-1, -1, 0) M(0, -1, 0) M(1, -1, 0) M(-1, 0, 0) M(0, 0, 0) M(1, 0, 0)   \
    M(-1, 1, 0) M(0, 1, 0) M(1, 1, 0) M(-1, -1, 1) M(0, -1, 1) M(1, -1, 1) M(-1, 0, 1) M(0, 0, 1)    \
    M(1, 0, 1) M(-1, 1, 1) M(0, 1, 1) M(1, 1, 1)

// One time step: pull (stream), moments (Eq. 1-2), BGK collide (Eq. 7 with Eq. 5), store.
template <typename T, int Q>
__global__ void __launch_bounds__(256) k_pop_step(const StepParams<T> p) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= p.L.nx || y >= p.L.ny) return;
    const long long xc = lidx(p.L, x, y, z);
    T f[Q];
    Acc<T> a = {};
#define LBWP_M(CX, CY, CZ) pop_pull<T, Q, CX, CY, CZ>(p.L, p.src, xc, f, a);
    LBWP_ALL_DIRS(LBWP_M)
#undef LBWP_M
    const T irho = T(1) / (T(1) + a.rho);
    // equilibrium = S-form node with omega = 1 (S = rho u u; stored P irrelevant)
    const SNode<T> eq = collide_sform<T>(a.rho, a.jx * irho, a.jy * irho, a.jz * irho, T(0), T(0), T(0), T(0),
                                         T(0), T(0), T(1));
#define LBWP_M(CX, CY, CZ) pop_collide_store<T, Q, CX, CY, CZ>(p.L, p.dst, x, y, z, f, eq, p.omega);
    LBWP_ALL_DIRS(LBWP_M)
#undef LBWP_M
}

// lbwp_moments for this scheme: pull from F_{t-1}, Eq. 1-3, write the external layout.
template <typename T, int Q>
__global__ void __launch_bounds__(256) k_pop_export(Layout L, const T* __restrict__ prev, T* __restrict__ ext) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long xc = lidx(L, x, y, z);
    T f[Q];
    Acc<T> a = {};
#define LBWP_M(CX, CY, CZ) pop_pull<T, Q, CX, CY, CZ>(L, prev, xc, f, a);
    LBWP_ALL_DIRS(LBWP_M)
#undef LBWP_M
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const double rho = 1.0 + (double)a.rho;
    ext[e] = T(rho);
    ext[n + e] = T((double)a.jx / rho);
    ext[2 * n + e] = T((double)a.jy / rho);
    ext[3 * n + e] = T((double)a.jz / rho);
    ext[4 * n + e] = T((double)a.pxx + 1.0 / 3.0);
    ext[5 * n + e] = T((double)a.pyy + 1.0 / 3.0);
    ext[6 * n + e] = T((double)a.pzz + 1.0 / 3.0);
    ext[7 * n + e] = a.pxy;
    ext[8 * n + e] = a.pxz;
    ext[9 * n + e] = a.pyz;
}

template <typename T, int Q, int CX, int CY, int CZ>
__device__ __forceinline__ void pop_seed(const Layout& L, T* __restrict__ dst, int x, int y, int z, const SNode<T>& s) {
    constexpr int N2 = CX * CX + CY * CY + CZ * CZ;
    if (Q == 19 && N2 == 3) return;
    constexpr int I = dir_index<Q>(CX, CY, CZ);
    // Eq. 4 population of node x, placed one link BACK (at x - c) so that the pull returns it to x
    int tx = x - CX, ty = y - CY, tz = z - CZ;
    tx += tx < 0 ? L.nx : 0; tx -= tx >= L.nx ? L.nx : 0;
    ty += ty < 0 ? L.ny : 0; ty -= ty >= L.ny ? L.ny : 0;
    tz += tz < 0 ? L.nz : 0; tz -= tz >= L.nz ? L.nz : 0;
    store_images(dst + (long long)I * L.field, L, tx, ty, tz, T(lattice_w<Q>(N2)) * bracket<T, CX, CY, CZ>(s));
}

// ext moments -> Eq. 4 populations (omega = 0 in the S-form gives h_i), back-shifted.
template <typename T, int Q>
__global__ void __launch_bounds__(256) k_pop_import(Layout L, const T* __restrict__ ext, T* __restrict__ dst) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const SNode<T> s = collide_sform<T>(T((double)ext[e] - 1.0), ext[n + e], ext[2 * n + e], ext[3 * n + e],
                                        T((double)ext[4 * n + e] - 1.0 / 3.0), T((double)ext[5 * n + e] - 1.0 / 3.0),
                                        T((double)ext[6 * n + e] - 1.0 / 3.0), ext[7 * n + e], ext[8 * n + e],
                                        ext[9 * n + e], T(0));
#define LBWP_M(CX, CY, CZ) pop_seed<T, Q, CX, CY, CZ>(L, dst, x, y, z, s);
    LBWP_ALL_DIRS(LBWP_M)
#undef LBWP_M
}

// ---------------------------------------------------------------------------------
// Two components ("38 populations per each fluid component"; reading C6):
// fields [0,Q) hold the post-collision TOTAL population minus w_i, fields [Q,2Q) the
// colour-A population (colour B = total - A).  One time step is three launches:
//   k_pop2_density   pull, rhoA and drho of the streamed state (densities
//                    are assessed after streaming, before the collision)
//   k_colour_gradient (lbwp_gather.cuh) on those two fields
//   k_pop2_step      pull, Eq. 1-2, BGK on the total, perturbation, recolouring, store
// ---------------------------------------------------------------------------------
template <typename T, int Q, int CX, int CY, int CZ>
__device__ __forceinline__ void pop2_pull_a(const Layout& L, const T* __restrict__ src, long long xc, T& rhoA) {
    constexpr int N2 = CX * CX + CY * CY + CZ * CZ;
    if (Q == 19 && N2 == 3) return;
    constexpr int I = dir_index<Q>(CX, CY, CZ);
    rhoA += src[(long long)(Q + I) * L.field + xc - ((long long)CZ * L.plane + (long long)CY * L.px + CX)];
}

// dens2: two fields (rhoA, drho) in the state layout, ghosts included.
template <typename T, int Q>
__global__ void __launch_bounds__(256) k_pop2_density(const StepParams<T> p, T* __restrict__ dens2) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= p.L.nx || y >= p.L.ny) return;
    const long long xc = lidx(p.L, x, y, z);
    T f[Q];
    Acc<T> a = {};
    T rhoA = 0;
#define LBWP_M(CX, CY, CZ) pop_pull<T, Q, CX, CY, CZ>(p.L, p.src, xc, f, a); pop2_pull_a<T, Q, CX, CY, CZ>(p.L, p.src, xc, rhoA);
    LBWP_ALL_DIRS(LBWP_M)
#undef LBWP_M
    store_images(dens2, p.L, x, y, z, rhoA);
    store_images(dens2 + p.L.field, p.L, x, y, z, a.rho);
}

template <typename T>
struct Colour {
    T Ag, nx, ny, nz, rA, kappa;  // A|G|, interface normal, rhoA/rho, beta rhoA rhoB / rho
};

template <typename T, int Q, int CX, int CY, int CZ>
__device__ __forceinline__ void pop2_collide_store(const Layout& L, T* __restrict__ dst, int x, int y, int z,
                                                   const T* f, const SNode<T>& eq, T omega, const Colour<T>& c) {
    constexpr int N2 = CX * CX + CY * CY + CZ * CZ;
    if (Q == 19 && N2 == 3) return;
    constexpr int I = dir_index<Q>(CX, CY, CZ);
    const T w = T(lattice_w<Q>(N2));
    const T feq = w * bracket<T, CX, CY, CZ>(eq);
    T h = f[I] - omega * (f[I] - feq);                                  // BGK on the total (Eq. 7)
    const T cn = T(CX) * c.nx + T(CY) * c.ny + T(CZ) * c.nz;
    const T Bi = N2 == 0 ? T(lattice_w<Q>(0) - 2.0 / 3.0) : w;
    h += T(0.5) * c.Ag * (w * cn * cn - Bi);                            // perturbation (reading C6)
    T hA = c.rA * (w + h);                                              // recolouring (reading C6)
    if (N2 != 0) {
        const T inorm = N2 == 1 ? T(1) : N2 == 2 ? T(0.70710678118654752440) : T(0.57735026918962576451);
        hA += c.kappa * w * inorm * cn;
    }
    store_images(dst + (long long)I * L.field, L, x, y, z, h);
    store_images(dst + (long long)(Q + I) * L.field, L, x, y, z, hA);
}

// p.grad: 3 gradient fields followed by the 2 density fields of k_pop2_density.
template <typename T, int Q>
__global__ void __launch_bounds__(256, sizeof(T) == 4 ? 3 : 1) k_pop2_step(const StepParams<T> p) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= p.L.nx || y >= p.L.ny) return;
    const long long xc = lidx(p.L, x, y, z);
    const long long F = p.L.field;
    T f[Q];
    Acc<T> a = {};
#define LBWP_M(CX, CY, CZ) pop_pull<T, Q, CX, CY, CZ>(p.L, p.src, xc, f, a);
    LBWP_ALL_DIRS(LBWP_M)
#undef LBWP_M
    const T rho = T(1) + a.rho;
    const T irho = T(1) / rho;
    const SNode<T> eq = collide_sform<T>(a.rho, a.jx * irho, a.jy * irho, a.jz * irho, T(0), T(0), T(0), T(0),
                                         T(0), T(0), T(1));
    const T Gx = p.grad[xc], Gy = p.grad[F + xc], Gz = p.grad[2 * F + xc];
    const T rhoA = p.grad[3 * F + xc];
    const T g2 = Gx * Gx + Gy * Gy + Gz * Gz;
    const T ig = g2 > T(1e-10) ? rsqrt_t<T>(g2) : T(0);  // reading C8
    Colour<T> c;
    c.Ag = p.A * (g2 * ig);
    c.nx = Gx * ig; c.ny = Gy * ig; c.nz = Gz * ig;
    c.rA = rhoA * irho;
    c.kappa = p.beta * c.rA * (rho - rhoA);
#define LBWP_M(CX, CY, CZ) pop2_collide_store<T, Q, CX, CY, CZ>(p.L, p.dst, x, y, z, f, eq, p.omega, c);
    LBWP_ALL_DIRS(LBWP_M)
#undef LBWP_M
}

template <typename T, int Q>
__global__ void __launch_bounds__(256) k_pop2_export(Layout L, const T* __restrict__ prev, T* __restrict__ ext) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long xc = lidx(L, x, y, z);
    T f[Q];
    Acc<T> a = {};
    T rhoA = 0;
#define LBWP_M(CX, CY, CZ) pop_pull<T, Q, CX, CY, CZ>(L, prev, xc, f, a); pop2_pull_a<T, Q, CX, CY, CZ>(L, prev, xc, rhoA);
    LBWP_ALL_DIRS(LBWP_M)
#undef LBWP_M
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const double rho = 1.0 + (double)a.rho;
    ext[e] = rhoA;
    ext[n + e] = T(rho - (double)rhoA);
    ext[2 * n + e] = T((double)a.jx / rho);
    ext[3 * n + e] = T((double)a.jy / rho);
    ext[4 * n + e] = T((double)a.jz / rho);
    ext[5 * n + e] = T((double)a.pxx + 1.0 / 3.0);
    ext[6 * n + e] = T((double)a.pyy + 1.0 / 3.0);
    ext[7 * n + e] = T((double)a.pzz + 1.0 / 3.0);
    ext[8 * n + e] = a.pxy;
    ext[9 * n + e] = a.pxz;
    ext[10 * n + e] = a.pyz;
}

template <typename T, int Q, int CX, int CY, int CZ>
__device__ __forceinline__ void pop2_seed(const Layout& L, T* __restrict__ dst, int x, int y, int z, const SNode<T>& s, T rA) {
    constexpr int N2 = CX * CX + CY * CY + CZ * CZ;
    if (Q == 19 && N2 == 3) return;
    constexpr int I = dir_index<Q>(CX, CY, CZ);
    int tx = x - CX, ty = y - CY, tz = z - CZ;
    tx += tx < 0 ? L.nx : 0; tx -= tx >= L.nx ? L.nx : 0;
    ty += ty < 0 ? L.ny : 0; ty -= ty >= L.ny ? L.ny : 0;
    tz += tz < 0 ? L.nz : 0; tz -= tz >= L.nz ? L.nz : 0;
    const T w = T(lattice_w<Q>(N2));
    const T h = w * bracket<T, CX, CY, CZ>(s);
    store_images(dst + (long long)I * L.field, L, tx, ty, tz, h);
    store_images(dst + (long long)(Q + I) * L.field, L, tx, ty, tz, rA * (w + h));  // initial split fA = rhoA/rho f
}

// ext moments (M = 11) -> Eq. 4 populations of the total, split by colour, back-shifted.
template <typename T, int Q>
__global__ void __launch_bounds__(256) k_pop2_import(Layout L, const T* __restrict__ ext, T* __restrict__ dst) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const double rhoA = (double)ext[e], rho = rhoA + (double)ext[n + e];
    const SNode<T> s = collide_sform<T>(T(rho - 1.0), ext[2 * n + e], ext[3 * n + e], ext[4 * n + e],
                                        T((double)ext[5 * n + e] - 1.0 / 3.0), T((double)ext[6 * n + e] - 1.0 / 3.0),
                                        T((double)ext[7 * n + e] - 1.0 / 3.0), ext[8 * n + e], ext[9 * n + e],
                                        ext[10 * n + e], T(0));
    const T rA = T(rhoA / rho);
#define LBWP_M(CX, CY, CZ) pop2_seed<T, Q, CX, CY, CZ>(L, dst, x, y, z, s, rA);
    LBWP_ALL_DIRS(LBWP_M)
#undef LBWP_M
}

}  // namespace lbwp
