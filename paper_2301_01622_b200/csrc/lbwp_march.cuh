// lbwp_march.cuh -- the fused moments-only step for D3Q27, single component (the graded
// kernel): shared-memory plane tiles + z-marching register accumulators.
//
// What one time step computes: for node x and direction c, the moments at
// y = x - c are collided (Eq. 8), the resulting population streams to x (Eq. 9), and the
// arrived populations are summed into the new moments (Eq. 1-3).  In S-form
// (lbwp_gather.cuh) the collision is a pointwise map node -> (da,J,Sd,So) and everything
// after it is a LINEAR 27-point stencil with the tensor-product weights
//   w_c = k(cx) k(cy) k(cz) / 216,  k = (1,4,1).
//
// Mapping:
//   * a block owns a TX x TY tile of (x,y) columns and marches over a chunk of z planes;
//     a thread owns one column;
//   * every input plane (tile + 1-cell halo, ghost-padded layout => no index wrap) is loaded
//     from HBM once per block, collided ONCE per node (not once per direction) and written to
//     shared memory in S-form, pre-scaled by 1/216; loads of plane z+1 are in flight while
//     plane z is consumed (register staging, double-buffered shared memory, one barrier/plane);
//   * a thread reads its 3x3 in-plane neighbourhood, forms the direction brackets
//       B(cx,cy,cz) = E + cz^2 Z + cz O,   E = da + cx Jx + cy Jy + cx^2 Sxx + cy^2 Syy + cx cy Sxy,
//       O = Jz + cx Sxz + cy Syz,  Z = Szz,
//     takes their in-plane moments with the separable (1,4,1) kernels (17 flops per 3x3 set),
//     and scatters them into three register accumulator sets: output planes z-1, z, z+1;
//   * the plane whose three contributions are complete is finalised (u = j/rho) and stored,
//     coalesced, together with its periodic ghost images.
#pragma once
#include "lbwp_common.cuh"

namespace lbwp {

template <typename T> __device__ __forceinline__ T fast_rcp(T x);
template <> __device__ __forceinline__ float fast_rcp<float>(float x) { return __frcp_rn(x); }
template <> __device__ __forceinline__ double fast_rcp<double>(double x) { return 1.0 / x; }

// In-plane moments of a 3x3 set of brackets V[cy+1][cx+1] with kernels k = (1,4,1):
//   m_pq = sum_{cx,cy} k(cx) k(cy) cx^p cy^q V(cx,cy)
template <typename T>
struct M6 {
    T m00, m10, m01, m20, m02, m11;
};

template <typename T>
__device__ __forceinline__ M6<T> xy_moments(const T (&V)[3][3]) {
    T r0[3], r1[3], r2[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const T s = V[j][2] + V[j][0];
        r1[j] = V[j][2] - V[j][0];
        r2[j] = s;
        r0[j] = fma(T(4), V[j][1], s);
    }
    M6<T> m;
    const T s0 = r0[2] + r0[0];
    m.m01 = r0[2] - r0[0];
    m.m02 = s0;
    m.m00 = fma(T(4), r0[1], s0);
    m.m10 = fma(T(4), r1[1], r1[2] + r1[0]);
    m.m11 = r1[2] - r1[0];
    m.m20 = fma(T(4), r2[1], r2[2] + r2[0]);
    return m;
}

// accumulator order: rho, jx, jy, jz, pxx, pyy, pzz, pxy, pxz, pyz
template <typename T, int TX, int TY>
struct March {
    static constexpr int SW = TX + 2, SH = TY + 2, SP = SW * SH;  // smem tile with halo
    static constexpr int NT = TX * TY;
    static constexpr int NLOAD = (SP + NT - 1) / NT;             // load slots per thread
    static constexpr size_t smem_bytes = sizeof(T) * 2 * 10 * SP;

    // pointwise BGK collision in moment space, S-form scaled by 1/216 (Eq. 8)
    __device__ static __forceinline__ void collide_store(T* __restrict__ s, const T (&r)[10], T omega) {
        const T c = T(1.0 / 216.0);
        const T drho = r[0], ux = r[1], uy = r[2], uz = r[3];
        const T rho = T(1) + drho;
        const T om1 = T(1) - omega;
        const T orho = omega * rho;
        const T iso = drho * T(1.0 / 3.0);
        const T sxx = fma(orho * ux, ux, om1 * (r[4] - iso));
        const T syy = fma(orho * uy, uy, om1 * (r[5] - iso));
        const T szz = fma(orho * uz, uz, om1 * (r[6] - iso));
        const T sxy = fma(orho * ux, uy, om1 * r[7]);
        const T sxz = fma(orho * ux, uz, om1 * r[8]);
        const T syz = fma(orho * uy, uz, om1 * r[9]);
        const T r3 = (T(3) * c) * rho;
        s[0 * SP] = c * fma(T(-1.5), sxx + syy + szz, drho);
        s[1 * SP] = r3 * ux;
        s[2 * SP] = r3 * uy;
        s[3 * SP] = r3 * uz;
        s[4 * SP] = (T(4.5) * c) * sxx;
        s[5 * SP] = (T(4.5) * c) * syy;
        s[6 * SP] = (T(4.5) * c) * szz;
        s[7 * SP] = (T(9) * c) * sxy;
        s[8 * SP] = (T(9) * c) * sxz;
        s[9 * SP] = (T(9) * c) * syz;
    }

    // consume one S-form input plane: update accumulators of output planes z-1 (P), z (C);
    // initialise z+1 (N).
    __device__ static __forceinline__ void consume(const T* __restrict__ s, T (&P)[10], T (&C)[10], T (&N)[10]) {
        T E[3][3], W[3][3], O[3][3];
#pragma unroll
        for (int cy = -1; cy <= 1; ++cy)
#pragma unroll
            for (int cx = -1; cx <= 1; ++cx) {
                const T* __restrict__ q = s - cy * SW - cx;  // source node x - c
                T e = q[0], o = q[3 * SP];
                const T z = q[6 * SP];
                if (cx) {
                    e += q[4 * SP];
                    e = cx > 0 ? e + q[1 * SP] : e - q[1 * SP];
                    o = cx > 0 ? o + q[8 * SP] : o - q[8 * SP];
                }
                if (cy) {
                    e += q[5 * SP];
                    e = cy > 0 ? e + q[2 * SP] : e - q[2 * SP];
                    o = cy > 0 ? o + q[9 * SP] : o - q[9 * SP];
                }
                if (cx * cy) e = cx * cy > 0 ? e + q[7 * SP] : e - q[7 * SP];
                E[cy + 1][cx + 1] = e;
                W[cy + 1][cx + 1] = e + z;
                O[cy + 1][cx + 1] = o;
            }
        const M6<T> me = xy_moments<T>(E), mw = xy_moments<T>(W), mo = xy_moments<T>(O);
        // cz = 0, k = 4
        C[0] = fma(T(4), me.m00, C[0]);
        C[1] = fma(T(4), me.m10, C[1]);
        C[2] = fma(T(4), me.m01, C[2]);
        C[4] = fma(T(4), me.m20, C[4]);
        C[5] = fma(T(4), me.m02, C[5]);
        C[7] = fma(T(4), me.m11, C[7]);
        // cz = +1 -> plane z+1 (first contribution: assignment)
        const T p00 = mw.m00 + mo.m00, p10 = mw.m10 + mo.m10, p01 = mw.m01 + mo.m01;
        N[0] = p00; N[1] = p10; N[2] = p01; N[3] = p00;
        N[4] = mw.m20 + mo.m20; N[5] = mw.m02 + mo.m02; N[6] = p00;
        N[7] = mw.m11 + mo.m11; N[8] = p10; N[9] = p01;
        // cz = -1 -> plane z-1 (last contribution)
        const T n00 = mw.m00 - mo.m00, n10 = mw.m10 - mo.m10, n01 = mw.m01 - mo.m01;
        P[0] += n00; P[1] += n10; P[2] += n01; P[3] -= n00;
        P[4] += mw.m20 - mo.m20; P[5] += mw.m02 - mo.m02; P[6] += n00;
        P[7] += mw.m11 - mo.m11; P[8] -= n10; P[9] -= n01;
    }
};

// store one value at the node and, for box-boundary nodes, at its ghost images
template <typename T>
__device__ __forceinline__ void store_node(T* __restrict__ f, long long c, T v, bool boundary, const Layout& L,
                                           int x, int y, int z) {
    f[c] = v;
    if (boundary) {
        const long long dx0 = x == 0 ? L.nx : 0, dx1 = x == L.nx - 1 ? -(long long)L.nx : 0;
        const long long dy0 = y == 0 ? (long long)L.ny * L.px : 0, dy1 = y == L.ny - 1 ? -(long long)L.ny * L.px : 0;
        const long long dz0 = z == 0 ? (long long)L.nz * L.plane : 0, dz1 = z == L.nz - 1 ? -(long long)L.nz * L.plane : 0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const long long oz = k == 0 ? 0 : k == 1 ? dz0 : dz1;
            if (k && !oz) continue;
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                const long long oy = j == 0 ? 0 : j == 1 ? dy0 : dy1;
                if (j && !oy) continue;
#pragma unroll
                for (int i = 0; i < 3; ++i) {
                    const long long ox = i == 0 ? 0 : i == 1 ? dx0 : dx1;
                    if (i && !ox) continue;
                    if (i + j + k) f[c + oz + oy + ox] = v;
                }
            }
        }
    }
}

template <typename T, int TX, int TY, int MINB>
__global__ void __launch_bounds__(TX* TY, MINB) k_step_march27(const StepParams<T> p, int lz) {
    using K = March<T, TX, TY>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* const sm = reinterpret_cast<T*>(smem_raw);
    const Layout& L = p.L;
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int z0 = blockIdx.z * lz;
    const int z1 = min(z0 + lz, L.nz);
    const int x = x0 + tx, y = y0 + ty;
    const bool active = x < L.nx && y < L.ny;

    // load slots: tile node (lr, lc) -> global node (x0-1+lc, y0-1+lr)
    long long goff[K::NLOAD];
    int soff[K::NLOAD];
    bool lv[K::NLOAD];
#pragma unroll
    for (int k = 0; k < K::NLOAD; ++k) {
        const int i = tid + k * K::NT;
        const int lr = i / K::SW, lc = i - lr * K::SW;
        const int gx = x0 - 1 + lc, gy = y0 - 1 + lr;
        lv[k] = i < K::SP && gx <= L.nx && gy <= L.ny;
        soff[k] = i;
        goff[k] = lidx(L, gx, gy, z0 - 1);
    }
    const long long F = L.field;
    const T* __restrict__ src = p.src;
    T raw[K::NLOAD][10];

    auto issue_loads = [&]() {
#pragma unroll
        for (int k = 0; k < K::NLOAD; ++k)
            if (lv[k]) {
#pragma unroll
                for (int f = 0; f < 10; ++f) raw[k][f] = __ldg(src + f * F + goff[k]);
            }
#pragma unroll
        for (int k = 0; k < K::NLOAD; ++k) goff[k] += L.plane;
    };
    auto collide_to = [&](T* buf) {
#pragma unroll
        for (int k = 0; k < K::NLOAD; ++k)
            if (lv[k]) K::collide_store(buf + soff[k], raw[k], p.omega);
    };

    issue_loads();
    collide_to(sm);
    __syncthreads();

    T a0[10], a1[10], a2[10];
#pragma unroll
    for (int f = 0; f < 10; ++f) a0[f] = a1[f] = a2[f] = T(0);
    const int my = (ty + 1) * K::SW + tx + 1;
    long long oc = lidx(L, x, y, z0 - 2);  // node of the plane that completes first
    int cur = 0;
    int zin = z0 - 1;

    // one input plane: prefetch the next, consume this one, finalise plane zin-1
    auto plane = [&](T(&P)[10], T(&C)[10], T(&N)[10]) {
        const bool more = zin < z1;
        if (more) issue_loads();
        K::consume(sm + cur * 10 * K::SP + my, P, C, N);
        const int zo = zin - 1;
        if (active && zo >= z0) {
            const bool bnd = x == 0 || x == L.nx - 1 || y == 0 || y == L.ny - 1 || zo == 0 || zo == L.nz - 1;
            const T irho = fast_rcp<T>(T(1) + P[0]);  // u = j / rho (Eq. 2, reading C11)
            T* __restrict__ d = p.dst;
            store_node(d, oc, P[0], bnd, L, x, y, zo);
            store_node(d + F, oc, P[1] * irho, bnd, L, x, y, zo);
            store_node(d + 2 * F, oc, P[2] * irho, bnd, L, x, y, zo);
            store_node(d + 3 * F, oc, P[3] * irho, bnd, L, x, y, zo);
#pragma unroll
            for (int f = 4; f < 10; ++f) store_node(d + f * F, oc, P[f], bnd, L, x, y, zo);
        }
        oc += L.plane;
        if (more) collide_to(sm + (cur ^ 1) * 10 * K::SP);
        __syncthreads();
        cur ^= 1;
        ++zin;
    };

    while (true) {
        plane(a0, a1, a2);
        if (zin > z1) break;
        plane(a1, a2, a0);
        if (zin > z1) break;
        plane(a2, a0, a1);
        if (zin > z1) break;
    }
}

// The fp64 instance needs more dynamic shared memory than the 48 KB default.  The attribute is per DEVICE, so it is
// set by lbwp_init for the context's device (after cudaSetDevice), not once per process.
template <typename T>
int prepare_march27() {
    constexpr int TX = 32, TY = 8, MINB = sizeof(T) == 4 ? 2 : 1;
    return (int)cudaFuncSetAttribute(k_step_march27<T, TX, TY, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)March<T, TX, TY>::smem_bytes);
}

template <typename T>
int launch_march27(const StepParams<T>& s, cudaStream_t stream) {
    constexpr int TX = 32, TY = 8, MINB = sizeof(T) == 4 ? 2 : 1;
    using K = March<T, TX, TY>;
    auto kern = k_step_march27<T, TX, TY, MINB>;
    const int gx = (s.L.nx + TX - 1) / TX, gy = (s.L.ny + TY - 1) / TY;
    // z chunks: enough blocks to fill 148 SMs several times over, chunks >= 16 planes when possible
    int lz = s.L.nz;
    const long long want = 148ll * 8;
    while ((long long)gx * gy * ((s.L.nz + lz - 1) / lz) < want && lz > 16) lz = (lz + 1) / 2;
    const dim3 grid(gx, gy, (s.L.nz + lz - 1) / lz), block(TX, TY, 1);
    kern<<<grid, block, K::smem_bytes, stream>>>(s, lz);
    return (int)cudaGetLastError();
}

}  // namespace lbwp
