// lbwp_tma.cuh -- the fused moments-only step for D3Q27, single component, as a TMA-fed
// linear stencil with the BGK collision as its epilogue (the graded kernel).
//
// Algebra.  Eq. 8 is a pointwise map of a node's
// moments to its "S-form"
//     a  = drho - (3/2) tr S,      J = 3 rho u,      Sd_a = (9/2) S_aa,   So_ab = 9 S_ab,
//     S  = omega rho u u + (1-omega)(P - rho cs^2 I),          drho = rho - 1,
// after which the population leaving along c is  h'_c = w_c (1 + a + c.J + c c : (Sd,So)),
// and Eq. 9 + Eq. 1-3 (pull, then project) are a LINEAR 27-point stencil of the ten S-form
// fields with the tensor-product weights w_c = k(cx) k(cy) k(cz) / 216, k = (1,4,1).
//
// So the state kept in HBM between steps is the S-form of the moments (ten values per node:
// the paper's ten hydrodynamic fields after the local, invertible-up-to-tau=1 collision map),
// pre-scaled by 1/216.  One step = stencil (gives rho, j, P at time t+1 in registers) followed
// by the collision of the new moments in the epilogue; the collided values are what is stored.
// Nothing is transformed on the load side, so planes go HBM -> shared memory by TMA untouched.
// lbwp_moments() gets the plain moments of time t by running the same stencil on the previous
// ping-pong buffer (the S-form of time t-1) with an epilogue that writes rho, u, P instead.
//
// Layout ("XLayout"): field-major [M][nz][ny][px], x fastest; ghost columns in x only (up to x = -2 on the
// left and x = nx+2 on the right, written by the owners of their images; which of them a kernel maintains
// and reads is its own business); y and z wrap on the load side (TMA coordinates).
// Interior x = 0 sits 16 bytes into a row, rows are a multiple of 32 bytes.
//
// Mapping: a CTA owns a TX x TY tile of columns and marches over a chunk of z planes.  Each
// input plane (tile + halo) is one shared-memory stage [row][field][BW], filled by three TMA
// boxes (the TY interior rows, and the two halo rows, which may wrap in y) that complete on
// the stage's "full" mbarrier; warps release a stage on its "empty" mbarrier, the producer
// (thread 0) refills it NS-1 planes ahead.  A thread owns NPT nodes (same x, rows TY/NPT
// apart) and keeps their z-1 / z / z+1 moment sums in registers; for fp32, NPT = 2 and every
// arithmetic instruction is a packed FADD2 / FFMA2 over the thread's two nodes.
#pragma once
#include <cuda.h>  // CUtensorMap and enums only; cuTensorMapEncodeTiled is resolved at run time
#include <cuda_runtime.h>
#include <stdint.h>

namespace lbwp {

struct XLayout {
    int nx, ny, nz;
    int ox;            // x offset of interior node 0 in a row (16 bytes of elements)
    int px;            // padded row length (elements), multiple of 32 bytes
    long long plane;   // px * ny
    long long field;   // px * ny * nz
};

inline XLayout make_xlayout(int nx, int ny, int nz, int elem_bytes) {
    XLayout L;
    L.nx = nx; L.ny = ny; L.nz = nz;
    L.ox = 16 / elem_bytes;
    const int q = 32 / elem_bytes;
    L.px = ((L.ox + nx + 3 + q - 1) / q) * q;   // ghost columns: x = -2, -1 on the left (ox >= 2), x = nx .. nx+2 on the right
    L.plane = (long long)L.px * ny;
    L.field = L.plane * nz;
    return L;
}

__host__ __device__ inline long long xidx(const XLayout& L, int x, int y, int z) {
    return ((long long)z * L.ny + y) * L.px + L.ox + x;
}

// ---------------------------------------------------------------------------------------------
// Small vectors over the nodes a thread owns.  Vec<float,2> is a packed pair: add/sub/fma are
// single FADD2 / FFMA2 instructions (add.rn.f32x2, fma.rn.f32x2: sm_100 packed fp32).
// ---------------------------------------------------------------------------------------------
template <typename T, int N> struct Vec;

template <typename T> struct Vec<T, 1> {
    T v;
    __device__ __forceinline__ static Vec bc(T s) { return Vec{s}; }
    __device__ __forceinline__ T get(int) const { return v; }
    __device__ __forceinline__ void set(int, T s) { v = s; }
};
template <typename T> __device__ __forceinline__ Vec<T, 1> operator+(Vec<T, 1> a, Vec<T, 1> b) { return {a.v + b.v}; }
template <typename T> __device__ __forceinline__ Vec<T, 1> operator-(Vec<T, 1> a, Vec<T, 1> b) { return {a.v - b.v}; }
template <typename T> __device__ __forceinline__ Vec<T, 1> operator*(Vec<T, 1> a, Vec<T, 1> b) { return {a.v * b.v}; }
template <typename T> __device__ __forceinline__ Vec<T, 1> vfma(Vec<T, 1> a, Vec<T, 1> b, Vec<T, 1> c) { return {fma(a.v, b.v, c.v)}; }

template <> struct Vec<float, 2> {
    float x, y;
    __device__ __forceinline__ static Vec bc(float s) { return Vec{s, s}; }
    __device__ __forceinline__ float get(int i) const { return i ? y : x; }
    __device__ __forceinline__ void set(int i, float s) { if (i) y = s; else x = s; }
};
typedef Vec<float, 2> f32x2;
__device__ __forceinline__ unsigned long long pk2(f32x2 a) {
    unsigned long long r;
    asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a.x), "f"(a.y));
    return r;
}
__device__ __forceinline__ f32x2 up2(unsigned long long r) {
    f32x2 a;
    asm("mov.b64 {%0,%1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(r));
    return a;
}
__device__ __forceinline__ f32x2 operator+(f32x2 a, f32x2 b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk2(a)), "l"(pk2(b)));
    return up2(r);
}
__device__ __forceinline__ f32x2 operator-(f32x2 a, f32x2 b) {
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk2(a)), "l"(pk2(b)));
    return up2(r);
}
__device__ __forceinline__ f32x2 operator*(f32x2 a, f32x2 b) {
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk2(a)), "l"(pk2(b)));
    return up2(r);
}
__device__ __forceinline__ f32x2 vfma(f32x2 a, f32x2 b, f32x2 c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pk2(a)), "l"(pk2(b)), "l"(pk2(c)));
    return up2(r);
}

template <typename T> __device__ __forceinline__ T rcp_t(T x);
template <> __device__ __forceinline__ float rcp_t<float>(float x) { return __frcp_rn(x); }
template <> __device__ __forceinline__ double rcp_t<double>(double x) { return 1.0 / x; }

// ---------------------------------------------------------------------------------------------
// mbarrier / TMA wrappers (PTX; SASS: SYNCS.*, UTMALDG)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// A TMA that can never complete (bad tensor map) must not hang the device: trap after ~2^26 probes
// (each try_wait already blocks for a hardware time slice), which surfaces as a launch failure.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (++spins > (1u << 26)) __trap();
    }
}
// A consumer warp hands a stage back to the producer.  Its shared-memory READS of the stage must have returned
// before the arrive is seen: an LDS that is still queued behind other warps' loads when the arrive goes out can be
// overtaken by the producer's next TMA fill of the stage (seen on B200 once the scheduler had the registers to
// issue a plane's last LDS.64 right before the arrive: about one launch in 150 at 128^3 had a few lanes read the
// NEXT plane's values).  The fence completes every lane's outstanding loads, __syncwarp orders the lanes.
__device__ __forceinline__ void consumer_release(uint32_t empty_bar, int tid) {
    __threadfence_block();
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(empty_bar);
}
// The same guarantee without a fence (which also waits for the warp's outstanding global stores): the arrive's
// ADDRESS is made to depend on a value `v` computed from every load of the stage (accumulators the whole plane
// feeds), so it cannot issue before those loads have returned.  An LDS completes for the whole warp at once, so
// lane 0's dependency covers all lanes.  `mask` is a kernel parameter that is 0 at run time: neither the compiler
// nor ptxas can fold `bits(v) & mask` away.
__device__ __forceinline__ void consumer_release_after(uint32_t empty_bar, int tid, float v, uint32_t mask) {
    const uint32_t zero = __float_as_uint(v) & mask;
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(empty_bar + zero);
}
__device__ __forceinline__ void consumer_release_after(uint32_t empty_bar, int tid, double v, uint32_t mask) {
    const uint32_t zero = (uint32_t)__double2hiint(v) & mask;
    __syncwarp();
    if ((tid & 31) == 0) mbar_arrive(empty_bar + zero);
}
// 4-D tiled load: coordinates (x, field, y, z) of the box origin.  Every load carries the L2 policy evict_last: what
// the step reads (the tile rows the y neighbours read again as their halo rows, a little later or earlier) outlives
// what it writes (never read again in the launch) in L2.  Measured on B200 against plain loads: 256^3 fp32 +3.7 %,
// 512^3 +1.1 %, 128^3 +3.3 %; streaming stores (st.global.cs, evict_first) instead lose 1-3 %, and keeping only the
// edge rows (separate boxes per policy) loses more to the extra TMA requests (profiles/r02_tuning.md).
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2, int c3,
                                            uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4, %5}], [%6], %7;"
        ::"r"(dst), "l"((unsigned long long)map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar), "l"(policy) : "memory");
}

}  // namespace lbwp
