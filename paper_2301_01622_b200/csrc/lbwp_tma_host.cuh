// lbwp_tma_host.cuh -- host side of the TMA step: tensor maps, grid sizing, launch; plus the
// pointwise import (moments -> S-form) and t = 0 export kernels of the XLayout state.
#pragma once
#include <cstdio>
#include <new>

#include "lbwp_tma_kernel.cuh"

namespace lbwp {

// ---- pointwise conversions (lbwp_init / lbwp_set_moments / lbwp_moments at t = 0; not per step) ----
// ext: dense [10][nz][ny][nx] moments (include/lbwp.h) -> sform: XLayout S-form (x ghosts included),
// raw: XLayout copy of the moments themselves (what lbwp_moments returns while no step was taken).
template <typename T, int Q>
__global__ void __launch_bounds__(256) k_tma_import(XLayout L, XLayout Lraw, const T* __restrict__ ext, T* __restrict__ sform,
                                                    T* __restrict__ raw, T omega) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const long long F = L.field, c = xidx(Lraw, x, y, z);
    T m[10];
#pragma unroll
    for (int f = 0; f < 10; ++f) { m[f] = ext[f * n + e]; raw[f * F + c] = m[f]; }
    // deviations taken in fp64 and rounded once; j = rho u
    T a[10];
    a[0] = T((double)m[0] - 1.0);
    for (int k = 0; k < 3; ++k) a[1 + k] = m[0] * m[1 + k];
    for (int k = 0; k < 3; ++k) a[4 + k] = T((double)m[4 + k] - 1.0 / 3.0);
    for (int k = 0; k < 3; ++k) a[7 + k] = m[7 + k];
    TmaStepParams<T> p;
    p.L = L; p.dst = sform; p.omega = omega; p.lz = 0;
    epilogue_node<T, EPI_SFORM, Q>(p, a, x, y, z);
}

template <typename T>
__global__ void __launch_bounds__(256) k_tma_export_raw(XLayout L, const T* __restrict__ raw, T* __restrict__ ext) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const long long F = L.field, c = xidx(L, x, y, z);
#pragma unroll
    for (int f = 0; f < 10; ++f) ext[f * n + e] = raw[f * F + c];
}

// ---- tensor maps -------------------------------------------------------------------------------
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline PFN_encodeTiled get_encode_tiled() {
    static PFN_encodeTiled fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (PFN_encodeTiled)p;
    }
    return fn;
}

// Tensor of one state buffer as TMA sees it: dims (x: px, field: M, y: ny, z: nz); box (bw, M, rows, 1).
template <typename T>
inline int make_state_map(CUtensorMap* out, const void* buf, const XLayout& L, int bw, int rows, int nfields = 10) {
    PFN_encodeTiled enc = get_encode_tiled();
    if (!enc) return -1;
    const cuuint64_t dims[4] = {(cuuint64_t)L.px, (cuuint64_t)nfields, (cuuint64_t)L.ny, (cuuint64_t)L.nz};
    const cuuint64_t strides[3] = {(cuuint64_t)L.field * sizeof(T), (cuuint64_t)L.px * sizeof(T),
                                   (cuuint64_t)L.plane * sizeof(T)};
    const cuuint32_t box[4] = {(cuuint32_t)bw, (cuuint32_t)nfields, (cuuint32_t)rows, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_L2_128B;   // none / 64 / 256 B measured within 1 %
    const CUresult r = enc(out, sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4,
                           const_cast<void*>(buf), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, promo,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : (int)r;
}

// ---- configured instances -------------------------------------------------------------------------
// One plan = one tile geometry (nodes per thread, tile x, tile y, stages; min CTAs per SM) bound to a
// context's two buffers.  Geometry choice: the widest tile that divides the box.
struct TmaPlanBase {
    XLayout L;       // layout of buffer 0
    XLayout Lb[2];   // per buffer: the x-paired fp32 kernel keeps buffer 1 one column to the right (TmaCfg)
    int lz = 0, gz = 0, resident = 0, grid = 0;
    char tag[32] = "";
    virtual ~TmaPlanBase() {}
    virtual int setup(const XLayout& L_, void* const buf[2]) = 0;
    // one pass: read the S-form in buffer `from`; epi = EPI_SFORM writes the S-form of the new moments
    // (XLayout), EPI_MOMENTS the new moments themselves (dense external layout)
    virtual int launch(int epi, int from, void* dst, double omega, cudaStream_t stream) const = 0;
};

// z chunking for `ctas` resident CTAs over `cols` tile columns.  Measured rules (B200, profiles/r02_tuning.md):
//  * several rounds of items: chunks of at most 32 planes.  Longer chunks let neighbouring CTAs drift apart until
//    their shared halo rows miss L2 (512^3: 37 GLUPS with 128-plane chunks, 57-68 with 16-32), and every new item
//    re-synchronises its neighbourhood;
//  * a launch whose items all run at once (one round) marches in lock-step from the start and tolerates chunks of
//    up to 128 planes (256^3 fp32: 2 x 64 items of 128 planes, 63.6 against 59.7 GLUPS with 9 x 64 items of 29;
//    384 planes in one go drift apart again: 49.9 against 64.2 at 384^3), and saves the halo planes: preferred
//    (10 % bonus) over a multi-round split of nominally equal cost.
// Cost = rounds x (planes + 2 halo planes).
inline void tma_choose_chunks(int nz, long long cols, int ctas, int* lz, int* gz) {
    const int LZMAX = 32, LZONE = 128;
    double best = 1e300;
    for (int g = 1; g <= nz; ++g) {
        const int l = (nz + g - 1) / g;
        if ((nz + l - 1) / l != g) continue;
        const long long rounds = (cols * g + ctas - 1) / ctas;
        if (l > (rounds == 1 ? LZONE : LZMAX) && g < nz) continue;
        const double cost = (double)rounds * (l + 2) * (rounds == 1 ? 0.9 : 1.0);
        if (cost < best - 1e-9) { best = cost; *lz = l; *gz = g; }
    }
}

template <typename T, typename C, int MINB>
struct TmaPlanT final : TmaPlanBase {
    CUtensorMap main_map[2], row_map[2];   // per ping-pong buffer

    template <int EPI>
    static auto kernel() { return k_step_tma27<T, C, EPI, MINB>; }

    int setup(const XLayout& L_, void* const buf[2]) override {
        L = L_;
        Lb[0] = Lb[1] = L;
        if (C::PX) Lb[1].ox += 1;
        snprintf(tag, sizeof(tag), "q%d_%dx%dx%d_s%d%s", C::Q, C::TX, C::TY, C::NPT, C::NS, C::PX ? "_px" : "");
        for (int k = 0; k < 2; ++k) {
            int rc = make_state_map<T>(&main_map[k], buf[k], L, C::BW, C::TY);
            if (rc) return rc;
            rc = make_state_map<T>(&row_map[k], buf[k], L, C::BW, 1);
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
        resident = per_sm * sms;
        const long long cols = (long long)(L.nx / C::TX) * (L.ny / C::TY);
        tma_choose_chunks(L.nz, cols, resident, &lz, &gz);
        const long long items = cols * gz;
        // one item per CTA: the hardware scheduler hands out items in order and keeps the frontier of
        // running items compact (a persistent grid with static striding measured 30 % slower at 512^3)
        grid = (int)items;
        return 0;
    }

    int launch(int epi, int from, void* dst, double omega, cudaStream_t stream) const override {
        TmaStepParams<T> p;
        p.L = Lb[from ^ 1]; p.dst = (T*)dst; p.omega = T(omega); p.lz = lz;   // EPI_SFORM writes the other buffer
        p.sh = (C::PX && from == 0) ? 1 : 0;
        if (epi == EPI_SFORM)
            kernel<EPI_SFORM>()<<<grid, C::NT + TMA_PRODUCER_THREADS, C::SMEM, stream>>>(main_map[from], row_map[from], p);
        else
            kernel<EPI_MOMENTS>()<<<grid, C::NT + TMA_PRODUCER_THREADS, C::SMEM, stream>>>(main_map[from], row_map[from], p);
        return (int)cudaGetLastError();
    }
};

// geometry lists: (nodes per thread, tile x, tile y, stages, min CTAs per SM, x-paired)
#define LBWP_F32_LIST(X) X(2, 128, 8, 3, 1, 1) X(2, 64, 8, 3, 1, 1)
#define LBWP_F64_LIST(X) X(1, 64, 8, 3, 1, 0) X(1, 32, 8, 3, 1, 0)

// first geometry of the dtype's list whose tile divides the box; nullptr if none does
template <typename T>
inline TmaPlanBase* make_tma_plan(int nx, int ny, int q);
#define LBWP_TRY(NPT, TX, TY, NS, MINB, PX)                                                                  \
    if (nx % TX == 0 && ny % TY == 0)                                                                        \
        return q == 27 ? (TmaPlanBase*)new (std::nothrow) TmaPlanT<float, TmaCfg<float, NPT, TX, TY, NS, 27, 1, PX>, MINB>() \
                       : (TmaPlanBase*)new (std::nothrow) TmaPlanT<float, TmaCfg<float, NPT, TX, TY, NS, 19, 1, PX>, MINB>();
template <> inline TmaPlanBase* make_tma_plan<float>(int nx, int ny, int q) { LBWP_F32_LIST(LBWP_TRY) return nullptr; }
#undef LBWP_TRY
#define LBWP_TRY(NPT, TX, TY, NS, MINB, PX)                                                                  \
    if (nx % TX == 0 && ny % TY == 0)                                                                        \
        return q == 27 ? (TmaPlanBase*)new (std::nothrow) TmaPlanT<double, TmaCfg<double, NPT, TX, TY, NS, 27, 1, PX>, MINB>() \
                       : (TmaPlanBase*)new (std::nothrow) TmaPlanT<double, TmaCfg<double, NPT, TX, TY, NS, 19, 1, PX>, MINB>();
template <> inline TmaPlanBase* make_tma_plan<double>(int nx, int ny, int q) { LBWP_F64_LIST(LBWP_TRY) return nullptr; }
#undef LBWP_TRY
#define LBWP_TRY(NPT, TX, TY, NS, MINB, PX) if (nx % TX == 0 && ny % TY == 0) return true;
inline bool tma_eligible_f32(int nx, int ny) { LBWP_F32_LIST(LBWP_TRY) return false; }
inline bool tma_eligible_f64(int nx, int ny) { LBWP_F64_LIST(LBWP_TRY) return false; }
#undef LBWP_TRY

}  // namespace lbwp
