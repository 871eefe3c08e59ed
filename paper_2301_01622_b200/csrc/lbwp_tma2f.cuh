// lbwp_tma2f.cuh -- two-component colour-gradient runs (reading C6), fused form (D3Q27 and D3Q19).
//
// State (two ping-pong buffers, XLayout, 16 fields each):
//   0..9   S-form of the total fluid after BGK only (x 1/216)      } written by the stencil kernel's epilogue
//   10     rA = rhoA / rho                                         } (the paper's eleven arrays, PAPER.md:75,
//   11     kappa = beta rhoA rhoB / rho (x 1/216)                  }  plus one derived from them)
//   12     gh = (A/2)|G| (x 1/216), G = (1/cs^2) sum_i w_i c_i phi(x + c_i), phi = 2 rA - 1
//   13..15 n = G/|G| (0 where |G|^2 <= 1e-10, reading C8)           } written by k_colour_normal
//
// One time step = k_step_tma27<NC = 3> (gather, perturbation and recolouring per direction, projection, BGK of the
// new moments in the epilogue: consume2f / store_state2f) + k_colour_normal (gradient of the new rA: one field read
// with its neighbours, four written).  Algorithmic traffic (16 + 12 + 1 + 4) x sizeof = 132 B fp32 per node and
// step, against 216 B of the split form (lbwp_tma2.cuh) and 88 B = 2 x 11 x sizeof if the gradient were taken
// inside the stencil kernel from a halo-2 tile (round-2 item).
// lbwp_moments: as in the single-component case, the moments of time t are the stencil of the previous buffer
// with an epilogue that writes (rhoA, rhoB, u, P).
#pragma once
#include "lbwp_tma_host.cuh"

namespace lbwp {

template <typename T>
struct Normal2Params {
    XLayout L;
    T* __restrict__ state;   // 16 fields; reads field 10, writes fields 12..15 (+ x ghost columns)
    T A;
};

// One thread per (x, y) column and ZC consecutive planes; the ZC + 2 planes of 3 x 3 rA values it needs sit in registers.
template <typename T, int Q, int ZC>
__global__ void __launch_bounds__(256) k_colour_normal(const Normal2Params<T> p) {
    const XLayout& L = p.L;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z0 = blockIdx.z * ZC;
    if (x >= L.nx || y >= L.ny) return;
    const long long F = L.field;
    const T* __restrict__ ra = p.state + 10 * F;
    // x neighbours come from the ghost columns the stencil epilogue maintains for rA; y and z wrap here (reading C13)
    const int ys[3] = {y == 0 ? L.ny - 1 : y - 1, y, y == L.ny - 1 ? 0 : y + 1};
    int off[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) off[j] = ys[j] * L.px + L.ox + x;
    auto load_plane = [&](int z, T (&f)[3][3]) {
        z = z < 0 ? z + L.nz : z;
        while (z >= L.nz) z -= L.nz;   // planes past a ragged last chunk are loaded (and ignored)
        const T* __restrict__ q = ra + (long long)z * L.plane;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            const T* __restrict__ qr = q + off[j];
            f[j][0] = qr[-1]; f[j][1] = qr[0]; f[j][2] = qr[1];
        }
    };
    // all ZC + 2 planes are requested before the first one is used: the pass is latency-bound otherwise
    // (9 loads in flight per thread gave 1.14 ms at 512^3 for 2.7 GB of traffic)
    T ph[ZC + 2][3][3];
#pragma unroll
    for (int k = 0; k < ZC + 2; ++k) load_plane(z0 - 1 + k, ph[k]);
#pragma unroll
    for (int k = 0; k < ZC; ++k) {
        const int z = z0 + k;
        if (z >= L.nz) break;
        T (&lo)[3][3] = ph[k];
        T (&mid)[3][3] = ph[k + 1];
        T (&hi)[3][3] = ph[k + 2];
        T gx = 0, gy = 0, gz = 0;   // G = 3 sum w c phi = 6 sum w c rA, because phi = 2 rA - 1 and sum w c = 0
#pragma unroll
        for (int cz = -1; cz <= 1; ++cz)
#pragma unroll
            for (int cy = -1; cy <= 1; ++cy)
#pragma unroll
                for (int cx = -1; cx <= 1; ++cx) {
                    const int n2 = cx * cx + cy * cy + cz * cz;
                    if (n2 == 0 || (Q == 19 && n2 == 3)) continue;
                    const T w = Q == 27 ? T(6.0 * (n2 == 1 ? 2.0 / 27.0 : n2 == 2 ? 1.0 / 54.0 : 1.0 / 216.0))
                                        : T(6.0 * (n2 == 1 ? 1.0 / 18.0 : 1.0 / 36.0));
                    const T f = cz < 0 ? lo[cy + 1][cx + 1] : cz == 0 ? mid[cy + 1][cx + 1] : hi[cy + 1][cx + 1];
                    if (cx) gx += T(cx) * w * f;
                    if (cy) gy += T(cy) * w * f;
                    if (cz) gz += T(cz) * w * f;
                }
        const T g2 = gx * gx + gy * gy + gz * gz;
        const T ig = g2 > T(1e-10) ? T(1) / sqrt(g2) : T(0);   // reading C8
        const T g = g2 * ig;
        T out[4];
        out[0] = (Q == 27 ? T(1.0 / 216.0) : T(1.0 / 36.0)) * T(0.5) * p.A * g;
        out[1] = gx * ig; out[2] = gy * ig; out[3] = gz * ig;
        T* __restrict__ d = p.state + 12 * F + (long long)z * L.plane + off[1];
#pragma unroll
        for (int f = 0; f < 4; ++f) d[f * F] = out[f];
        if (x == 0 || x == L.nx - 1) {
            T* __restrict__ gd = x == 0 ? d + L.nx : d - L.nx;
#pragma unroll
            for (int f = 0; f < 4; ++f) gd[f * F] = out[f];
        }
    }
}

// dense external moments [11][nz][ny][nx] (rhoA, rhoB, u, P) -> state fields 0..11 (and a plain copy for t = 0)
template <typename T, int Q>
__global__ void __launch_bounds__(256) k_tma2f_import(XLayout L, const T* __restrict__ ext, T* __restrict__ state,
                                                      T* __restrict__ raw, T omega, T beta) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const long long F = L.field, c = xidx(L, x, y, z);
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
    store_state2f<T, Q>(L, state, a, omega, beta, x, y, z);
}

template <typename T>
__global__ void __launch_bounds__(256) k_tma2f_export_raw(XLayout L, const T* __restrict__ raw, T* __restrict__ ext) {
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
template <typename T, int Q> struct Tma2fGeom;
template <int Q> struct Tma2fGeom<float, Q> { using C = TmaCfg<float, 2, 64, 8, 3, Q, 3>; };
template <int Q> struct Tma2fGeom<double, Q> { using C = TmaCfg<double, 1, 32, 8, 3, Q, 3>; };

struct Tma2fPlanBase {
    virtual ~Tma2fPlanBase() {}
    virtual int setup(const XLayout& L_, void* const buf[2]) = 0;
    virtual int stencil(int epi, int from, void* dst, double omega, double beta, cudaStream_t stream) const = 0;
    virtual int normals(void* state, double A, cudaStream_t stream) const = 0;
    virtual int import_state(const void* ext, void* state, void* raw, double omega, double beta, cudaStream_t stream) const = 0;
};

template <typename T, int Q>
struct Tma2fPlan final : Tma2fPlanBase {
    using C = typename Tma2fGeom<T, Q>::C;
    XLayout L;
    CUtensorMap main_map[2], row_map[2];
    int lz = 0, gz = 0, grid = 0;

    static bool eligible(int nx, int ny) { return nx % C::TX == 0 && ny % C::TY == 0; }
    template <int EPI>
    static auto kernel() { return k_step_tma27<T, C, EPI, 1>; }

    int setup(const XLayout& L_, void* const buf[2]) override {
        L = L_;
        for (int k = 0; k < 2; ++k) {
            int rc = make_state_map<T>(&main_map[k], buf[k], L, C::BW, C::TY, C::M);
            if (rc) return rc;
            rc = make_state_map<T>(&row_map[k], buf[k], L, C::BW, 1, C::M);
            if (rc) return rc;
        }
        cudaError_t e = cudaFuncSetAttribute(kernel<EPI_SFORM>(), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(kernel<EPI_MOMENTS>(), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
        if (e != cudaSuccess) return (int)e;
        int per_sm = 0, dev = 0, sms = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel<EPI_SFORM>(), C::NT + TMA_PRODUCER_THREADS, C::SMEM) != cudaSuccess || per_sm < 1)
            per_sm = 1;
        const long long cols = (long long)(L.nx / C::TX) * (L.ny / C::TY);
        tma_choose_chunks(L.nz, cols, per_sm * sms, &lz, &gz);
        grid = (int)(cols * gz);
        return 0;
    }

    // stencil pass from buffer `from`: EPI_SFORM -> state fields 0..11 of dst, EPI_MOMENTS -> dense moments in dst
    int stencil(int epi, int from, void* dst, double omega, double beta, cudaStream_t stream) const override {
        TmaStepParams<T> p;
        p.L = L; p.dst = (T*)dst; p.omega = T(omega); p.lz = lz; p.beta = T(beta);
        if (epi == EPI_SFORM) kernel<EPI_SFORM>()<<<grid, C::NT + TMA_PRODUCER_THREADS, C::SMEM, stream>>>(main_map[from], row_map[from], p);
        else kernel<EPI_MOMENTS>()<<<grid, C::NT + TMA_PRODUCER_THREADS, C::SMEM, stream>>>(main_map[from], row_map[from], p);
        return (int)cudaGetLastError();
    }

    // gradient pass on one state buffer: fields 12..15 from field 10
    int normals(void* state, double A, cudaStream_t stream) const override {
        constexpr int ZC = 4;
        Normal2Params<T> a;
        a.L = L; a.state = (T*)state; a.A = T(A);
        const int bx = L.nx >= 128 ? 128 : (L.nx >= 64 ? 64 : 32), by = 256 / bx;
        const dim3 b(bx, by, 1), g((L.nx + bx - 1) / bx, (L.ny + by - 1) / by, (L.nz + ZC - 1) / ZC);
        k_colour_normal<T, Q, ZC><<<g, b, 0, stream>>>(a);
        return (int)cudaGetLastError();
    }

    int import_state(const void* ext, void* state, void* raw, double omega, double beta, cudaStream_t stream) const override {
        const dim3 b(32, 8, 1), g((L.nx + 31) / 32, (L.ny + 7) / 8, L.nz);
        k_tma2f_import<T, Q><<<g, b, 0, stream>>>(L, (const T*)ext, (T*)state, (T*)raw, T(omega), T(beta));
        return (int)cudaGetLastError();
    }
};

}  // namespace lbwp
