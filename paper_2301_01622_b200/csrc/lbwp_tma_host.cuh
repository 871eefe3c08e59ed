// lbwp_tma_host.cuh -- host side of the TMA step: tensor maps, grid sizing, launch; plus the
// pointwise import (moments -> S-form) and t = 0 export kernels of the XLayout state.
#pragma once
#include "lbwp_tma_kernel.cuh"

namespace lbwp {

// ---- pointwise conversions (lbwp_init / lbwp_set_moments / lbwp_moments at t = 0; not per step) ----
// ext: dense [10][nz][ny][nx] moments (include/lbwp.h) -> sform: XLayout S-form (x ghosts included),
// raw: XLayout copy of the moments themselves (what lbwp_moments returns while no step was taken).
template <typename T>
__global__ void __launch_bounds__(256) k_tma_import(XLayout L, const T* __restrict__ ext, T* __restrict__ sform,
                                                    T* __restrict__ raw, T omega) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= L.nx || y >= L.ny) return;
    const long long n = (long long)L.nx * L.ny * L.nz;
    const long long e = ((long long)z * L.ny + y) * L.nx + x;
    const long long F = L.field, c = xidx(L, x, y, z);
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
    epilogue_node<T, EPI_SFORM>(p, a, x, y, z);
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

// Tensor of one state buffer as TMA sees it: dims (x: px, field: 10, y: ny, z: nz); box (bw, 10, rows, 1).
template <typename T>
inline int make_state_map(CUtensorMap* out, const void* buf, const XLayout& L, int bw, int rows) {
    PFN_encodeTiled enc = get_encode_tiled();
    if (!enc) return -1;
    const cuuint64_t dims[4] = {(cuuint64_t)L.px, 10, (cuuint64_t)L.ny, (cuuint64_t)L.nz};
    const cuuint64_t strides[3] = {(cuuint64_t)L.field * sizeof(T), (cuuint64_t)L.px * sizeof(T),
                                   (cuuint64_t)L.plane * sizeof(T)};
    const cuuint32_t box[4] = {(cuuint32_t)bw, 10, (cuuint32_t)rows, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = enc(out, sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4,
                           const_cast<void*>(buf), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : (int)r;
}

// ---- one configured instance ---------------------------------------------------------------------
template <typename T> struct TmaInst;
template <> struct TmaInst<float> { using C = TmaCfg<float, 2, 64, 8, 3>; static constexpr int MINB = 2; };
template <> struct TmaInst<double> { using C = TmaCfg<double, 1, 32, 8, 3>; static constexpr int MINB = 2; };

template <typename T>
struct TmaPlan {
    using C = typename TmaInst<T>::C;
    XLayout L;
    CUtensorMap main_map[2], row_map[2];   // per ping-pong buffer
    int lz = 0, gz = 0, resident = 0;

    static bool eligible(int nx, int ny, int nz) { return nx % C::TX == 0 && ny % C::TY == 0 && nz >= 1; }

    template <int EPI>
    static auto kernel() { return k_step_tma27<T, C, EPI, TmaInst<T>::MINB>; }

    int setup(const XLayout& L_, void* const buf[2]) {
        L = L_;
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
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel<EPI_SFORM>(), C::NT, C::SMEM) != cudaSuccess || per_sm < 1)
            per_sm = 1;
        resident = per_sm * sms;
        // z chunking: minimise waves x (planes per chunk + 2 halo planes); DESIGN.md "Grid sizing"
        const long long cols = (long long)(L.nx / C::TX) * (L.ny / C::TY);
        double best = 1e300;
        for (int g = 1; g <= L.nz; ++g) {
            const int l = (L.nz + g - 1) / g;
            if ((L.nz + l - 1) / l != g) continue;
            const long long blocks = cols * g;
            const long long waves = (blocks + resident - 1) / resident;
            const double cost = (double)waves * (l + 2) * (blocks < resident ? 1.0 : 1.0);
            if (cost < best - 1e-9) { best = cost; lz = l; gz = g; }
        }
        return 0;
    }

    // one step: read the S-form in buffer `from`, write into `dst` (S-form of the new moments, or the
    // new moments themselves for EPI_MOMENTS)
    template <int EPI>
    int launch(int from, T* dst, T omega, cudaStream_t stream) const {
        TmaStepParams<T> p;
        p.L = L; p.dst = dst; p.omega = omega; p.lz = lz;
        const dim3 grid(L.nx / C::TX, L.ny / C::TY, gz), block(C::NT, 1, 1);
        kernel<EPI>()<<<grid, block, C::SMEM, stream>>>(main_map[from], row_map[from], p);
        return (int)cudaGetLastError();
    }
};

}  // namespace lbwp
