// lbwp_tma2.cuh -- two-component colour-gradient runs (reading C6) in the paper's own SPLIT form
// ("collision ... store post-collision hydro fields ... separate streaming kernel"), with the
// streaming kernel being the TMA stencil of lbwp_tma*.cuh.
//
//   pass A  k_colour_collide (pointwise + 26-neighbour gradient of phi; a thread marches 8 planes in z and keeps
//           the phi neighbourhood in registers):
//           R = (rhoA, drho, j, dP_aa, P_ab, phi)  ->  S15 = (S-form with the perturbation folded in, rA, K, R0)
//   pass B  k_step_tma27<NC = 2>: linear stencil of S15 (consume2c), raw sums stored back into R.
//
// R is the state between steps (12 fields, what lbwp_moments reads); S15 is scratch (15 fields).
// Algorithmic traffic: A reads 12 + writes 15, B reads 15 + writes 12 fields = 54 x sizeof per node and step
// (216 B fp32), against the 2 x 11 x sizeof of a fully fused step: the fused version is the round-2 item.
#pragma once
#include "lbwp_gather.cuh"
#include "lbwp_tma_host.cuh"

namespace lbwp {

template <typename T>
struct Colour2Params {
    XLayout L;
    const T* __restrict__ raw;   // 12 fields, XLayout (ghost columns unused: this pass wraps its indices)
    T* __restrict__ s15;         // 15 fields, XLayout, x ghost columns written here
    T omega, A, beta;
};

// One thread per (x, y) column, ZC consecutive planes: the 3 x 3 x 3 neighbourhood of phi lives in registers
// and only its top plane (9 values) is loaded per node.
template <typename T, int Q, int ZC>
__global__ void __launch_bounds__(256) k_colour_collide(const Colour2Params<T> p) {
    const XLayout& L = p.L;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z0 = blockIdx.z * ZC;
    if (x >= L.nx || y >= L.ny) return;
    const long long F = L.field;
    const T* __restrict__ r = p.raw;
    const T* __restrict__ phi = r + 11 * F;
    const int xs[3] = {x == 0 ? L.nx - 1 : x - 1, x, x == L.nx - 1 ? 0 : x + 1};
    const int ys[3] = {y == 0 ? L.ny - 1 : y - 1, y, y == L.ny - 1 ? 0 : y + 1};
    int off[3][3];   // in-plane offsets of the nine columns (periodic, reading C13)
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int i = 0; i < 3; ++i) off[j][i] = ys[j] * L.px + L.ox + xs[i];
    auto load_plane = [&](int z, T (&f)[3][3]) {
        z = z < 0 ? z + L.nz : (z >= L.nz ? z - L.nz : z);
        const T* __restrict__ q = phi + (long long)z * L.plane;
#pragma unroll
        for (int j = 0; j < 3; ++j)
#pragma unroll
            for (int i = 0; i < 3; ++i) f[j][i] = q[off[j][i]];
    };
    T ph[3][3][3];   // [plane z-1, z, z+1][y][x]
    load_plane(z0 - 1, ph[0]);
    load_plane(z0, ph[1]);
    const T c = Q == 27 ? T(1.0 / 216.0) : T(1.0 / 36.0);
#pragma unroll
    for (int k = 0; k < ZC; ++k) {
        const int z = z0 + k;
        if (z >= L.nz) break;
        T (&lo)[3][3] = ph[k % 3];
        T (&mid)[3][3] = ph[(k + 1) % 3];
        T (&hi)[3][3] = ph[(k + 2) % 3];
        load_plane(z + 1, hi);
        // gradient of the phase field, G = (1/cs^2) sum_i w_i c_i phi(x + c_i)  (reading C6)
        T gx = 0, gy = 0, gz = 0;
#pragma unroll
        for (int cz = -1; cz <= 1; ++cz)
#pragma unroll
            for (int cy = -1; cy <= 1; ++cy)
#pragma unroll
                for (int cx = -1; cx <= 1; ++cx) {
                    const int n2 = cx * cx + cy * cy + cz * cz;
                    if (n2 == 0 || (Q == 19 && n2 == 3)) continue;
                    const T w = T(3.0 * lattice_w<Q>(n2));
                    const T f = cz < 0 ? lo[cy + 1][cx + 1] : cz == 0 ? mid[cy + 1][cx + 1] : hi[cy + 1][cx + 1];
                    if (cx) gx += T(cx) * w * f;
                    if (cy) gy += T(cy) * w * f;
                    if (cz) gz += T(cz) * w * f;
                }
        const long long c0 = (long long)z * L.plane + off[1][1];
        const T rhoA = r[c0], drho = r[F + c0];
        const T rho = T(1) + drho, irho = T(1) / rho;
        const T jx = r[2 * F + c0], jy = r[3 * F + c0], jz = r[4 * F + c0];
        SNode<T> n = collide_sform<T>(drho, jx * irho, jy * irho, jz * irho, r[5 * F + c0], r[6 * F + c0], r[7 * F + c0],
                                      r[8 * F + c0], r[9 * F + c0], r[10 * F + c0], p.omega);
        const T g2 = gx * gx + gy * gy + gz * gz;
        const T ig = g2 > T(1e-10) ? rsqrt_t<T>(g2) : T(0);   // reading C8
        const T g = g2 * ig;
        const T nx = gx * ig, ny = gy * ig, nz = gz * ig;
        const T Ag = p.A * g;
        // perturbation: S_tot = S + (A/9)|G| n n, drho' = drho - (A/3)|G|, rest population + (A/3)|G|
        n.da -= Ag * T(1.0 / 3.0) + Ag * T(1.5 / 9.0);
        n.Sxx += T(0.5) * Ag * nx * nx;
        n.Syy += T(0.5) * Ag * ny * ny;
        n.Szz += T(0.5) * Ag * nz * nz;
        n.Sxy += Ag * nx * ny;
        n.Sxz += Ag * nx * nz;
        n.Syz += Ag * ny * nz;
        const T rA = rhoA * irho;
        const T kappa = p.beta * rA * (rho - rhoA);   // beta rhoA rhoB / rho
        T out[15];
        out[0] = c * n.da;
        out[1] = c * n.Jx; out[2] = c * n.Jy; out[3] = c * n.Jz;
        out[4] = c * n.Sxx; out[5] = c * n.Syy; out[6] = c * n.Szz;
        out[7] = c * n.Sxy; out[8] = c * n.Sxz; out[9] = c * n.Syz;
        out[10] = rA;
        out[11] = c * kappa * nx; out[12] = c * kappa * ny; out[13] = c * kappa * nz;
        out[14] = Ag * T(1.0 / 3.0);
        T* __restrict__ d = p.s15 + c0;
#pragma unroll
        for (int f = 0; f < 15; ++f) d[f * F] = out[f];
        if (x == 0 || x == L.nx - 1) {   // x ghost column for the TMA boxes of pass B
            T* __restrict__ gdst = x == 0 ? d + L.nx : d - L.nx;
#pragma unroll
            for (int f = 0; f < 15; ++f) gdst[f * F] = out[f];
        }
    }
}

// dense external moments [11][nz][ny][nx] (rhoA, rhoB, u, P) <-> R
template <typename T>
__global__ void __launch_bounds__(256) k_tma2_import(XLayout L, const T* __restrict__ ext, T* __restrict__ raw) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const long long F = L.field, c = xidx(L, x, y, z);
    const double ra = (double)ext[e], rb = (double)ext[n + e];
    const double rho = ra + rb;
    raw[c] = T(ra);
    raw[F + c] = T(rho - 1.0);
    for (int k = 0; k < 3; ++k) raw[(2 + k) * F + c] = T(rho * (double)ext[(2 + k) * n + e]);
    for (int k = 0; k < 3; ++k) raw[(5 + k) * F + c] = T((double)ext[(5 + k) * n + e] - 1.0 / 3.0);
    for (int k = 0; k < 3; ++k) raw[(8 + k) * F + c] = ext[(8 + k) * n + e];
    raw[11 * F + c] = T((ra - rb) / rho);
}

template <typename T>
__global__ void __launch_bounds__(256) k_tma2_export(XLayout L, const T* __restrict__ raw, T* __restrict__ ext) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const long long F = L.field, c = xidx(L, x, y, z);
    const double ra = (double)raw[c], rho = 1.0 + (double)raw[F + c];
    ext[e] = T(ra);
    ext[n + e] = T(rho - ra);
    for (int k = 0; k < 3; ++k) ext[(2 + k) * n + e] = T((double)raw[(2 + k) * F + c] / rho);   // u = j / rho (C11)
    for (int k = 0; k < 3; ++k) ext[(5 + k) * n + e] = T((double)raw[(5 + k) * F + c] + 1.0 / 3.0);
    for (int k = 0; k < 3; ++k) ext[(8 + k) * n + e] = raw[(8 + k) * F + c];
}

// ---- host side: one two-component plan per dtype ----------------------------------------------------
template <typename T, int Q> struct Tma2Geom;
template <int Q> struct Tma2Geom<float, Q> { using C = TmaCfg<float, 2, 64, 8, 3, Q, 2>; };
template <int Q> struct Tma2Geom<double, Q> { using C = TmaCfg<double, 1, 32, 8, 3, Q, 2>; };

struct Tma2PlanBase {
    virtual ~Tma2PlanBase() {}
    virtual int setup(const XLayout& L_, void* s15) = 0;
    virtual int step(void* raw, void* s15, double omega, double A, double beta, cudaStream_t stream) const = 0;
};

template <typename T, int Q>
struct Tma2Plan final : Tma2PlanBase {
    using C = typename Tma2Geom<T, Q>::C;
    XLayout L;
    CUtensorMap main_map, row_map;   // over the S15 scratch buffer
    int lz = 0, gz = 0, grid = 0;

    static bool eligible(int nx, int ny) { return nx % C::TX == 0 && ny % C::TY == 0; }
    static auto kernel() { return k_step_tma27<T, C, EPI_SFORM, 1>; }

    int setup(const XLayout& L_, void* s15) override {
        L = L_;
        int rc = make_state_map<T>(&main_map, s15, L, C::BW, C::TY, C::M);
        if (rc) return rc;
        rc = make_state_map<T>(&row_map, s15, L, C::BW, 1, C::M);
        if (rc) return rc;
        cudaError_t e = cudaFuncSetAttribute(kernel(), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
        if (e != cudaSuccess) return (int)e;
        int per_sm = 0, dev = 0, sms = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel(), C::NT + TMA_PRODUCER_THREADS, C::SMEM) != cudaSuccess || per_sm < 1)
            per_sm = 1;
        const long long cols = (long long)(L.nx / C::TX) * (L.ny / C::TY);
        tma_choose_chunks(L.nz, cols, per_sm * sms, &lz, &gz);
        grid = (int)(cols * gz);
        return 0;
    }

    // one time step: collide R -> S15, then stream S15 -> R
    int step(void* raw, void* s15, double omega, double A, double beta, cudaStream_t stream) const override {
        Colour2Params<T> a;
        a.L = L; a.raw = (const T*)raw; a.s15 = (T*)s15; a.omega = T(omega); a.A = T(A); a.beta = T(beta);
        constexpr int ZC = 8;
        // rows as long as the box allows: 27 field streams of 128-byte pieces ran at 4.2 TB/s, see profiles/
        const int bx = L.nx >= 128 ? 128 : (L.nx >= 64 ? 64 : 32), by = 256 / bx;
        const dim3 b(bx, by, 1), g((L.nx + bx - 1) / bx, (L.ny + by - 1) / by, (L.nz + ZC - 1) / ZC);
        k_colour_collide<T, Q, ZC><<<g, b, 0, stream>>>(a);
        TmaStepParams<T> p;
        p.L = L; p.dst = (T*)raw; p.omega = T(omega); p.lz = lz;
        kernel()<<<grid, C::NT + TMA_PRODUCER_THREADS, C::SMEM, stream>>>(main_map, row_map, p);
        return (int)cudaGetLastError();
    }
};

}  // namespace lbwp
