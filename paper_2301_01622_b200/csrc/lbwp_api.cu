// lbwp_api.cu -- the C ABI of include/lbwp.h over the sm_100a kernels.
// Host logic only: argument checks, buffer ownership, ping-pong bookkeeping
// ("Flip-Flop") and kernel selection.  No CPU fallback exists.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include "../../include/lbwp.h"
#include "lbwp_common.cuh"
#include "lbwp_convert.cuh"
#include "lbwp_diag.cuh"
#include "lbwp_gather.cuh"
#include "lbwp_march.cuh"
#include "lbwp_pop.cuh"
#include "lbwp_tma_host.cuh"
#include "lbwp_tma2.cuh"
#include "lbwp_tma2g.cuh"
#include "lbwp_contact.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

// every entry point works on the context's device and leaves the caller's current device as it found it
struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != dev) ok = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

#define CU(call)                                                                               \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess)                                                                 \
            return fail(e_ == cudaErrorMemoryAllocation ? LBWP_ENOMEM : LBWP_ECUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                               \
    } while (0)

bool params_ok(const lbwp_params* p) {
    if (!p || p->struct_size != (int32_t)sizeof(lbwp_params)) return false;
    if (p->lattice != 19 && p->lattice != 27) return false;
    if (p->dtype != LBWP_F32 && p->dtype != LBWP_F64) return false;
    if (p->ncomp != 1 && p->ncomp != 2) return false;
    if (p->scheme != LBWP_MOMENTS && p->scheme != LBWP_POPULATIONS) return false;
    if (p->kernel < LBWP_KERNEL_AUTO || p->kernel > LBWP_KERNEL_TMA_SPLIT) return false;
    if (p->nx < 1 || p->ny < 1 || p->nz < 1) return false;
    if ((long long)p->nx * p->ny * p->nz > (1ll << 31)) return false;
    if (p->nz > 65535 || (p->ny + 7) / 8 > 65535) return false;   // the pointwise kernels put z (and y / 8) in gridDim.z (.y)
    if (!(p->tau > 0.5)) return false;  // also rejects NaN
    if ((p->buf[0] == nullptr) != (p->buf[1] == nullptr)) return false;
    if (p->A_h != 0.0 && !(p->ncomp == 2 && p->scheme == LBWP_MOMENTS && p->h_c > 0.0)) return false;   // also rejects NaN h_c
    if (p->A_h != p->A_h) return false;
    return true;
}

int elem_bytes(const lbwp_params* p) { return p->dtype == LBWP_F32 ? 4 : 8; }
int num_moments(const lbwp_params* p) { return p->ncomp == 1 ? 10 : 11; }
int state_fields(const lbwp_params* p) {
    return p->scheme == LBWP_MOMENTS ? num_moments(p) : p->ncomp * p->lattice;
}


bool tma_eligible(const lbwp_params* p) {
    if (p->scheme == LBWP_MOMENTS && p->ncomp == 2)
        return p->dtype == LBWP_F32 ? lbwp::Tma2gPlan<float, 27>::eligible(p->nx, p->ny)
                                    : lbwp::Tma2gPlan<double, 27>::eligible(p->nx, p->ny);
    if (!(p->scheme == LBWP_MOMENTS && p->ncomp == 1)) return false;
    return p->dtype == LBWP_F32 ? lbwp::tma_eligible_f32(p->nx, p->ny) : lbwp::tma_eligible_f64(p->nx, p->ny);
}

// two-component TMA runs: fused form unless the split form is asked for
bool tma2_fused(const lbwp_params* p) { return p->ncomp == 2 && p->kernel != LBWP_KERNEL_TMA_SPLIT; }

// kernel variant a context with these params runs (LBWP_KERNEL_AUTO resolved); 0 if not built
int choose_variant(const lbwp_params* p) {
    if (p->A_h != 0.0) {   // near-contact force: a fix-up pass behind the fused two-component TMA step, or the generic kernels
        if (p->kernel == LBWP_KERNEL_AUTO || p->kernel == LBWP_KERNEL_TMA) {
            if (tma_eligible(p)) return LBWP_KERNEL_TMA;
            return p->kernel == LBWP_KERNEL_AUTO ? LBWP_KERNEL_GATHER : 0;
        }
        return p->kernel == LBWP_KERNEL_GATHER ? LBWP_KERNEL_GATHER : 0;
    }
    const bool march_ok = p->scheme == LBWP_MOMENTS && p->ncomp == 1 && p->lattice == 27;
    switch (p->kernel) {
        case LBWP_KERNEL_AUTO: return tma_eligible(p) ? LBWP_KERNEL_TMA : march_ok ? LBWP_KERNEL_MARCH : LBWP_KERNEL_GATHER;
        case LBWP_KERNEL_TMA: return tma_eligible(p) ? LBWP_KERNEL_TMA : 0;
        case LBWP_KERNEL_TMA_SPLIT: return (p->ncomp == 2 && tma_eligible(p)) ? LBWP_KERNEL_TMA : 0;
        case LBWP_KERNEL_MARCH: return march_ok ? LBWP_KERNEL_MARCH : 0;
        default: return LBWP_KERNEL_GATHER;
    }
}

}  // namespace

struct lbwp_ctx {
    lbwp_params P;
    lbwp::Layout L;
    int M = 0, nfields = 0, esize = 0;
    void* buf[2] = {nullptr, nullptr};
    bool owns = false;
    void* grad = nullptr;     // ncomp==2: colour gradient scratch, 3 fields
    void* staging = nullptr;  // dense external-layout device buffer for host <-> device I/O
    void* diag = nullptr;     // lbwp_diagnostics: block partials, probe coordinates, results
    int cur = 0;
    int64_t steps = 0;
    cudaStream_t stream = nullptr;
    int variant = LBWP_KERNEL_GATHER;
    int launches_per_step = 1;
    char name[64] = "";
    virtual ~lbwp_ctx() {}
    virtual int step_once() = 0;
    virtual int import_dense(const void* dev_ext) = 0;
    virtual int export_dense(void* dev_ext) = 0;
    // geometry of z planes in the state buffers, in elements: field stride, plane stride, offset of logical plane 0,
    // number of state fields; and the buffer that holds the CURRENT state (halo exchange, lbwp_halo_*)
    virtual void plane_geometry(long long* field, long long* plane, long long* z0off, int* nf) const = 0;
    virtual void* state_buffer() const { return buf[cur]; }
};

namespace {

dim3 node_grid(const lbwp::Layout& L, dim3 b) { return dim3((L.nx + b.x - 1) / b.x, (L.ny + b.y - 1) / b.y, L.nz); }

template <typename T>
struct Ctx final : lbwp_ctx {
    lbwp::StepParams<T> sp(int from, int to) const {
        lbwp::StepParams<T> s;
        s.L = L;
        s.src = (const T*)buf[from];
        s.dst = (T*)buf[to];
        s.grad = (const T*)grad;
        s.omega = T(1.0 / P.tau);
        s.A = T(P.A);
        s.beta = T(P.beta);
        if (P.A_h != 0.0) {
            s.force = (const T*)grad + 3 * L.field;   // scratch: 3 gradient + 3 force fields
            s.A_h = T(P.A_h);
            s.h_c = T(P.h_c);
        }
        return s;
    }

    template <int Q, int NC>
    int step_moments(const lbwp::StepParams<T>& s) {
        const dim3 b(32, 8, 1), g = node_grid(L, b);
        if (NC == 2) lbwp::k_colour_gradient<T, Q><<<g, b, 0, stream>>>(s, (T*)grad);
        if (NC == 1 && Q == 27 && variant == LBWP_KERNEL_MARCH) return lbwp::launch_march27<T>(s, stream);
        if (NC == 2 && s.force) {
            lbwp::k_near_contact<T, Q><<<g, b, 0, stream>>>(s, (const T*)grad, (T*)grad + 3 * L.field);
            lbwp::k_step_gather<T, Q, 2, 1><<<g, b, 0, stream>>>(s);
            return 0;
        }
        lbwp::k_step_gather<T, Q, NC><<<g, b, 0, stream>>>(s);
        return 0;
    }

    // two-component population step (lbwp_pop.cuh): grad = 3 gradient fields + 2 density fields
    template <int Q>
    void step_pop2(const lbwp::StepParams<T>& s) {
        const dim3 b(32, 8, 1), g = node_grid(L, b);
        T* dens2 = (T*)grad + 3 * L.field;
        lbwp::k_pop2_density<T, Q><<<g, b, 0, stream>>>(s, dens2);
        lbwp::StepParams<T> d = s;
        d.src = dens2;
        lbwp::k_colour_gradient<T, Q><<<g, b, 0, stream>>>(d, (T*)grad);
        lbwp::k_pop2_step<T, Q><<<g, b, 0, stream>>>(s);
    }

    int step_once() override {
        const lbwp::StepParams<T> s = sp(cur, cur ^ 1);
        const dim3 b(32, 8, 1), g = node_grid(L, b);
        if (P.scheme == LBWP_POPULATIONS && P.ncomp == 2) {
            if (P.lattice == 27) step_pop2<27>(s); else step_pop2<19>(s);
        } else if (P.scheme == LBWP_POPULATIONS) {
            if (P.lattice == 27) lbwp::k_pop_step<T, 27><<<g, b, 0, stream>>>(s);
            else lbwp::k_pop_step<T, 19><<<g, b, 0, stream>>>(s);
        } else {
            int rc = 0;
            if (P.lattice == 27) rc = P.ncomp == 1 ? step_moments<27, 1>(s) : step_moments<27, 2>(s);
            else rc = P.ncomp == 1 ? step_moments<19, 1>(s) : step_moments<19, 2>(s);
            if (rc) return fail(LBWP_ECUDA, "march kernel launch: %s", cudaGetErrorString((cudaError_t)rc));
        }
        CU(cudaGetLastError());
        cur ^= 1;
        ++steps;
        return LBWP_OK;
    }

    int import_dense(const void* ext) override {
        const dim3 b(32, 8, 1), g = node_grid(L, b);
        steps = 0;
        if (P.scheme == LBWP_POPULATIONS) {
            // seed F_{-1} in buf[1], then one collide pass gives F_0 in buf[0] (lbwp_pop.cuh)
            if (P.ncomp == 2) {
                if (P.lattice == 27) lbwp::k_pop2_import<T, 27><<<g, b, 0, stream>>>(L, (const T*)ext, (T*)buf[1]);
                else lbwp::k_pop2_import<T, 19><<<g, b, 0, stream>>>(L, (const T*)ext, (T*)buf[1]);
            } else if (P.lattice == 27) lbwp::k_pop_import<T, 27><<<g, b, 0, stream>>>(L, (const T*)ext, (T*)buf[1]);
            else lbwp::k_pop_import<T, 19><<<g, b, 0, stream>>>(L, (const T*)ext, (T*)buf[1]);
            CU(cudaGetLastError());
            cur = 1;
            int rc = step_once();
            steps = 0;
            return rc;
        }
        cur = 0;
        if (P.ncomp == 1) lbwp::k_import_moments<T, 1><<<g, b, 0, stream>>>(L, (const T*)ext, (T*)buf[0]);
        else lbwp::k_import_moments<T, 2><<<g, b, 0, stream>>>(L, (const T*)ext, (T*)buf[0]);
        CU(cudaGetLastError());
        return LBWP_OK;
    }

    void plane_geometry(long long* field, long long* plane, long long* z0off, int* nf) const override {
        *field = L.field; *plane = L.plane; *z0off = L.plane; *nf = nfields;   // one ghost plane below logical plane 0
    }
    int export_dense(void* ext) override {
        const dim3 b(32, 8, 1), g = node_grid(L, b);
        if (P.scheme == LBWP_POPULATIONS) {
            if (P.ncomp == 2) {
                if (P.lattice == 27) lbwp::k_pop2_export<T, 27><<<g, b, 0, stream>>>(L, (const T*)buf[cur ^ 1], (T*)ext);
                else lbwp::k_pop2_export<T, 19><<<g, b, 0, stream>>>(L, (const T*)buf[cur ^ 1], (T*)ext);
            } else if (P.lattice == 27) lbwp::k_pop_export<T, 27><<<g, b, 0, stream>>>(L, (const T*)buf[cur ^ 1], (T*)ext);
            else lbwp::k_pop_export<T, 19><<<g, b, 0, stream>>>(L, (const T*)buf[cur ^ 1], (T*)ext);
        } else if (P.ncomp == 1) {
            lbwp::k_export_moments<T, 1><<<g, b, 0, stream>>>(L, (const T*)buf[cur], (T*)ext);
        } else {
            lbwp::k_export_moments<T, 2><<<g, b, 0, stream>>>(L, (const T*)buf[cur], (T*)ext);
        }
        CU(cudaGetLastError());
        return LBWP_OK;
    }
};

// Context of the TMA variant: buf[] hold the S-form in XLayout (lbwp_tma.cuh).  buf[cur] = S-form of
// the moments at the current time t; buf[cur^1] = S-form of time t-1 (t >= 1), or the plain moments
// themselves (t = 0), which is what lbwp_moments needs in either case.
template <typename T>
struct TmaCtx final : lbwp_ctx {
    lbwp::TmaPlanBase* planp = nullptr;
    lbwp::XLayout X;
    ~TmaCtx() override { delete planp; }

    int prepare() {
        planp = lbwp::make_tma_plan<T>(X.nx, X.ny, P.lattice);
        if (!planp) return fail(LBWP_ENOMEM, "no TMA plan");
        int rc = planp->setup(X, buf);
        if (rc) return fail(rc < 0 ? LBWP_EUNSUPPORTED : LBWP_ECUDA, "TMA plan setup failed (%d): %s", rc,
                            rc < 0 ? "cuTensorMapEncodeTiled not available" : "tensor map / attribute error");
        return LBWP_OK;
    }
    int step_once() override {
        int rc = planp->launch(lbwp::EPI_SFORM, cur, buf[cur ^ 1], 1.0 / P.tau, stream);
        if (rc) return fail(LBWP_ECUDA, "tma step launch: %s", cudaGetErrorString((cudaError_t)rc));
        cur ^= 1;
        ++steps;
        return LBWP_OK;
    }
    int import_dense(const void* ext) override {
        const dim3 b(32, 8, 1), g((X.nx + 31) / 32, (X.ny + 7) / 8, X.nz);
        steps = 0;
        cur = 0;
        if (P.lattice == 27) lbwp::k_tma_import<T, 27><<<g, b, 0, stream>>>(planp->Lb[0], planp->Lb[1], (const T*)ext, (T*)buf[0], (T*)buf[1], T(1.0 / P.tau));
        else lbwp::k_tma_import<T, 19><<<g, b, 0, stream>>>(planp->Lb[0], planp->Lb[1], (const T*)ext, (T*)buf[0], (T*)buf[1], T(1.0 / P.tau));
        CU(cudaGetLastError());
        return LBWP_OK;
    }
    void plane_geometry(long long* field, long long* plane, long long* z0off, int* nf) const override {
        *field = X.field; *plane = X.plane; *z0off = 0; *nf = 10;
    }
    int export_dense(void* ext) override {
        if (steps == 0) {
            const dim3 b(32, 8, 1), g((X.nx + 31) / 32, (X.ny + 7) / 8, X.nz);
            lbwp::k_tma_export_raw<T><<<g, b, 0, stream>>>(planp->Lb[cur ^ 1], (const T*)buf[cur ^ 1], (T*)ext);
            CU(cudaGetLastError());
            return LBWP_OK;
        }
        int rc = planp->launch(lbwp::EPI_MOMENTS, cur ^ 1, ext, 1.0 / P.tau, stream);
        if (rc) return fail(LBWP_ECUDA, "tma export launch: %s", cudaGetErrorString((cudaError_t)rc));
        return LBWP_OK;
    }
};

// Two-component TMA variant (lbwp_tma2.cuh): buf[0] = S15 scratch, buf[1] = R, the state (12 of 15 fields used).
template <typename T>
struct Tma2Ctx final : lbwp_ctx {
    lbwp::Tma2PlanBase* planp = nullptr;
    lbwp::XLayout X;
    ~Tma2Ctx() override { delete planp; }

    int prepare() {
        planp = P.lattice == 27 ? (lbwp::Tma2PlanBase*)new (std::nothrow) lbwp::Tma2Plan<T, 27>()
                                : (lbwp::Tma2PlanBase*)new (std::nothrow) lbwp::Tma2Plan<T, 19>();
        if (!planp) return fail(LBWP_ENOMEM, "no two-component TMA plan");
        int rc = planp->setup(X, buf[0]);
        if (rc) return fail(rc < 0 ? LBWP_EUNSUPPORTED : LBWP_ECUDA, "two-component TMA plan setup failed (%d)", rc);
        return LBWP_OK;
    }
    int step_once() override {
        int rc = planp->step(buf[1], buf[0], 1.0 / P.tau, P.A, P.beta, stream);
        if (rc) return fail(LBWP_ECUDA, "two-component step launch: %s", cudaGetErrorString((cudaError_t)rc));
        ++steps;
        return LBWP_OK;
    }
    int import_dense(const void* ext) override {
        const dim3 b(32, 8, 1), g((X.nx + 31) / 32, (X.ny + 7) / 8, X.nz);
        steps = 0;
        lbwp::k_tma2_import<T><<<g, b, 0, stream>>>(X, (const T*)ext, (T*)buf[1]);
        CU(cudaGetLastError());
        return LBWP_OK;
    }
    void plane_geometry(long long* field, long long* plane, long long* z0off, int* nf) const override {
        *field = X.field; *plane = X.plane; *z0off = 0; *nf = 12;
    }
    void* state_buffer() const override { return buf[1]; }   // R; buf[0] is the scratch of the collide pass
    int export_dense(void* ext) override {
        const dim3 b(32, 8, 1), g((X.nx + 31) / 32, (X.ny + 7) / 8, X.nz);
        lbwp::k_tma2_export<T><<<g, b, 0, stream>>>(X, (const T*)buf[1], (T*)ext);
        CU(cudaGetLastError());
        return LBWP_OK;
    }
};

// Fused two-component TMA variant (lbwp_tma2g.cuh): two ping-pong state buffers of 11 fields, one launch per step.
// buf[cur] = state of time t; buf[cur^1] = state of time t-1 (t >= 1) or the plain moments (t = 0), which lbwp_moments needs.
template <typename T>
struct Tma2gCtx final : lbwp_ctx {
    lbwp::Tma2gPlanBase* planp = nullptr;
    lbwp::XLayout X;
    int sms = 148;
    ~Tma2gCtx() override { delete planp; }

    int prepare() {
        planp = P.lattice == 27 ? (lbwp::Tma2gPlanBase*)new (std::nothrow) lbwp::Tma2gPlan<T, 27>()
                                : (lbwp::Tma2gPlanBase*)new (std::nothrow) lbwp::Tma2gPlan<T, 19>();
        if (!planp) return fail(LBWP_ENOMEM, "no fused two-component TMA plan");
        int rc = planp->setup(X, buf);
        if (rc) return fail(rc < 0 ? LBWP_EUNSUPPORTED : LBWP_ECUDA, "fused two-component TMA plan setup failed (%d)", rc);
        if (P.A_h != 0.0) {   // min and max of rA per box, written by k_contact_scan (the layout's box grid is the same for both buffers)
            cudaError_t e = cudaMalloc(&grad, (size_t)2 * lbwp::contact_boxes(X).count() * sizeof(T));
            if (e != cudaSuccess) return fail(LBWP_ENOMEM, "cudaMalloc(near-contact box ranges): %s", cudaGetErrorString(e));
            e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, P.device);
            if (e != cudaSuccess) return fail(LBWP_ECUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
        }
        return LBWP_OK;
    }
    // near-contact force (lbwp_contact.cuh): Guo's forcing applied to the collided moments of buffer b, in place
    int contact_fixup(int b) {
        if (P.A_h == 0.0) return LBWP_OK;
        lbwp::ContactParams<T> cp;
        cp.L = planp->Lb[b]; cp.state = (T*)buf[b];
        cp.omega = T(1.0 / P.tau); cp.A_h = T(P.A_h); cp.h_c = T(P.h_c);
        using namespace lbwp;
        const ContactBoxes B = contact_boxes(cp.L);
        const dim3 blk(CONTACT_BX, CONTACT_BY, 1);
        const T* ra = (const T*)buf[b] + 10 * cp.L.field;
        const int zb = B.count() >= 64 * sms ? 8 : 2;           // boxes along z per CTA of the scan
        const dim3 gs(B.nbx, B.nby, (B.nbz + zb - 1) / zb);
        if (zb == 8) k_contact_scan<T, 8><<<gs, blk, 0, stream>>>(cp.L, B, ra, (T*)grad);
        else k_contact_scan<T, 2><<<gs, blk, 0, stream>>>(cp.L, B, ra, (T*)grad);
        const int split = B.count() >= 64 * sms ? 1 : CONTACT_BZ;   // 128^3: 2048 boxes, 512^3: 131072
        // large grids: more CTAs than fit at once, so that the block scheduler evens out the SMs (measured: 32 per SM
        // 2.89 ms per step at 512^3 against 2.92 with 8); small grids: what is resident at once (128^3: 4 per SM
        // 0.1047 ms per step, 8: 0.1056, 16: 0.1088, 32: 0.114)
        const int gf = (int)std::min<long long>((long long)B.count() * split, (split == 1 ? 32 : 4) * sms);
        if (P.lattice == 27) k_contact_fixup<T, 27><<<gf, blk, 0, stream>>>(cp, B, (const T*)grad, split);
        else k_contact_fixup<T, 19><<<gf, blk, 0, stream>>>(cp, B, (const T*)grad, split);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail(LBWP_ECUDA, "near-contact fix-up launch: %s", cudaGetErrorString(e));
        return LBWP_OK;
    }
    int step_once() override {
        int rc = planp->stencil(lbwp::EPI_SFORM, cur, buf[cur ^ 1], 1.0 / P.tau, P.A, P.beta, stream);
        if (rc) return fail(LBWP_ECUDA, "fused two-component step launch: %s", cudaGetErrorString((cudaError_t)rc));
        cur ^= 1;
        ++steps;
        return contact_fixup(cur);
    }
    int import_dense(const void* ext) override {
        steps = 0;
        cur = 0;
        int rc = planp->import_state(ext, buf[0], buf[1], 1.0 / P.tau, stream);
        if (rc) return fail(LBWP_ECUDA, "import launch: %s", cudaGetErrorString((cudaError_t)rc));
        return contact_fixup(0);
    }
    void plane_geometry(long long* field, long long* plane, long long* z0off, int* nf) const override {
        *field = X.field; *plane = X.plane; *z0off = 0; *nf = 11;
    }
    int export_dense(void* ext) override {
        if (steps == 0) {
            const dim3 b(32, 8, 1), g((X.nx + 31) / 32, (X.ny + 7) / 8, X.nz);
            lbwp::k_tma2g_export_raw<T><<<g, b, 0, stream>>>(planp->Lb[cur ^ 1], (const T*)buf[cur ^ 1], (T*)ext);
            CU(cudaGetLastError());
            return LBWP_OK;
        }
        int rc = planp->stencil(lbwp::EPI_MOMENTS, cur ^ 1, ext, 1.0 / P.tau, P.A, P.beta, stream);
        if (rc) return fail(LBWP_ECUDA, "fused two-component export launch: %s", cudaGetErrorString((cudaError_t)rc));
        return LBWP_OK;
    }
};

size_t dense_bytes(const lbwp_ctx* c) { return (size_t)c->M * c->L.nx * c->L.ny * c->L.nz * c->esize; }

int load_moments(lbwp_ctx* c, const void* moments, int on_device) {
    if (!moments) return fail(LBWP_EINVAL, "moments is NULL");
    const void* dev = moments;
    if (!on_device) {
        if (!c->staging) CU(cudaMalloc(&c->staging, dense_bytes(c)));
        CU(cudaMemcpyAsync(c->staging, moments, dense_bytes(c), cudaMemcpyHostToDevice, c->stream));
        dev = c->staging;
    }
    int rc = c->import_dense(dev);
    if (rc) return rc;
    CU(cudaStreamSynchronize(c->stream));
    return LBWP_OK;
}

}  // namespace

extern "C" {

size_t lbwp_state_bytes(const lbwp_params* p) {
    if (!params_ok(p)) return 0;
    const int variant = choose_variant(p);
    if (variant == 0) return 0;
    if (variant == LBWP_KERNEL_TMA) {
        const lbwp::XLayout X = lbwp::make_xlayout(p->nx, p->ny, p->nz, elem_bytes(p));
        return (size_t)(p->ncomp == 2 ? (tma2_fused(p) ? 11 : 15) : 10) * (size_t)X.field * (size_t)elem_bytes(p);
    }
    const lbwp::Layout L = lbwp::make_layout(p->nx, p->ny, p->nz, elem_bytes(p));
    return (size_t)state_fields(p) * (size_t)L.field * (size_t)elem_bytes(p);
}

int lbwp_num_moments(const lbwp_params* p) { return params_ok(p) ? num_moments(p) : 0; }

int lbwp_init(const lbwp_params* p, const void* moments, int moments_on_device, lbwp_ctx** out) {
    if (!out) return fail(LBWP_EINVAL, "out is NULL");
    if (!params_ok(p)) return fail(LBWP_EINVAL, "invalid lbwp_params (lattice 19|27, dtype, ncomp 1|2, sizes >= 1, tau > 0.5, A_h only with ncomp 2 moments and h_c > 0, struct_size)");
    if (!moments) return fail(LBWP_EINVAL, "moments is NULL");
    const int variant = choose_variant(p);
    if (variant == 0)
        return fail(LBWP_EUNSUPPORTED, "kernel %d is not built for this combination (MARCH: D3Q27 single-component moments; TMA: moments "
                    "scheme with nx %% 64 (fp32) or 32 (fp64) == 0 and ny %% 8 == 0; TMA_SPLIT: two-component only; A_h != 0: AUTO or GATHER)", p->kernel);
    int ndev = 0;
    CU(cudaGetDeviceCount(&ndev));
    if (p->device < 0 || p->device >= ndev) return fail(LBWP_EINVAL, "device %d out of range (%d devices)", p->device, ndev);
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, p->device));
    if (prop.major != 10)
        return fail(LBWP_EUNSUPPORTED, "device %d is sm_%d%d; this library is built for sm_100a only", p->device, prop.major, prop.minor);
    DeviceGuard guard(p->device);
    if (!guard.ok) return fail(LBWP_ECUDA, "cudaSetDevice(%d) failed", p->device);

    lbwp_ctx* c = nullptr;
    if (variant == LBWP_KERNEL_TMA) {
        const lbwp::XLayout X = lbwp::make_xlayout(p->nx, p->ny, p->nz, elem_bytes(p));
        if (tma2_fused(p)) {
            if (p->dtype == LBWP_F32) { auto* t = new (std::nothrow) Tma2gCtx<float>(); if (t) t->X = X; c = t; }
            else { auto* t = new (std::nothrow) Tma2gCtx<double>(); if (t) t->X = X; c = t; }
        } else if (p->ncomp == 2) {
            if (p->dtype == LBWP_F32) { auto* t = new (std::nothrow) Tma2Ctx<float>(); if (t) t->X = X; c = t; }
            else { auto* t = new (std::nothrow) Tma2Ctx<double>(); if (t) t->X = X; c = t; }
        } else if (p->dtype == LBWP_F32) { auto* t = new (std::nothrow) TmaCtx<float>(); if (t) t->X = X; c = t; }
        else { auto* t = new (std::nothrow) TmaCtx<double>(); if (t) t->X = X; c = t; }
    } else {
        c = p->dtype == LBWP_F32 ? (lbwp_ctx*)new (std::nothrow) Ctx<float>() : (lbwp_ctx*)new (std::nothrow) Ctx<double>();
    }
    if (!c) return fail(LBWP_ENOMEM, "host allocation failed");
    c->P = *p;
    c->esize = elem_bytes(p);
    c->L = lbwp::make_layout(p->nx, p->ny, p->nz, c->esize);
    c->M = num_moments(p);
    c->nfields = state_fields(p);
    c->stream = (cudaStream_t)p->stream;
    const size_t bytes = lbwp_state_bytes(p);
    int rc = LBWP_OK;
    auto bail = [&](int code) { lbwp_destroy(c); return code; };
    if (p->buf[0]) {
        if (((uintptr_t)p->buf[0] | (uintptr_t)p->buf[1]) & 255) return bail(fail(LBWP_EINVAL, "buf[] must be 256-byte aligned"));
        c->buf[0] = p->buf[0];
        c->buf[1] = p->buf[1];
    } else {
        c->owns = true;
        for (int k = 0; k < 2; ++k) {
            cudaError_t e = cudaMalloc(&c->buf[k], bytes);
            if (e != cudaSuccess) return bail(fail(LBWP_ENOMEM, "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e)));
        }
    }
    if (p->scheme == LBWP_MOMENTS && p->ncomp == 2 && variant != LBWP_KERNEL_TMA) {
        const bool nc = p->A_h != 0.0;
        cudaError_t e = cudaMalloc(&c->grad, (size_t)(nc ? 6 : 3) * c->L.field * c->esize);
        if (e != cudaSuccess) return bail(fail(LBWP_ENOMEM, "cudaMalloc(grad): %s", cudaGetErrorString(e)));
        c->launches_per_step = nc ? 3 : 2;
    }
    if (p->scheme == LBWP_POPULATIONS && p->ncomp == 2) {
        const size_t gb = (size_t)5 * c->L.field * c->esize;  // 3 gradient + 2 density fields
        cudaError_t e = cudaMalloc(&c->grad, gb);
        if (e != cudaSuccess) return bail(fail(LBWP_ENOMEM, "cudaMalloc(grad): %s", cudaGetErrorString(e)));
        e = cudaMemsetAsync(c->grad, 0, gb, c->stream);
        if (e != cudaSuccess) return bail(fail(LBWP_ECUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e)));
        c->launches_per_step = 3;
    }
    // ghost cells and padding start defined (padding is never read by a node update)
    for (int k = 0; k < 2; ++k) {
        cudaError_t e = cudaMemsetAsync(c->buf[k], 0, bytes, c->stream);
        if (e != cudaSuccess) return bail(fail(LBWP_ECUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e)));
    }
    c->variant = variant;
    if (variant == LBWP_KERNEL_MARCH) {
        const int e = p->dtype == LBWP_F32 ? lbwp::prepare_march27<float>() : lbwp::prepare_march27<double>();
        if (e) return bail(fail(LBWP_ECUDA, "march kernel attribute: %s", cudaGetErrorString((cudaError_t)e)));
    }
    if (variant == LBWP_KERNEL_TMA) {
        if (tma2_fused(p)) {
            rc = p->dtype == LBWP_F32 ? static_cast<Tma2gCtx<float>*>(c)->prepare() : static_cast<Tma2gCtx<double>*>(c)->prepare();
            c->launches_per_step = p->A_h != 0.0 ? 3 : 1;   // + the two kernels of the near-contact fix-up pass
        } else if (p->ncomp == 2) {
            rc = p->dtype == LBWP_F32 ? static_cast<Tma2Ctx<float>*>(c)->prepare() : static_cast<Tma2Ctx<double>*>(c)->prepare();
            c->launches_per_step = 2;
        } else {
            rc = p->dtype == LBWP_F32 ? static_cast<TmaCtx<float>*>(c)->prepare() : static_cast<TmaCtx<double>*>(c)->prepare();
        }
        if (rc) return bail(rc);
    }
    snprintf(c->name, sizeof(c->name), "%s%d_%s%s",
             p->scheme == LBWP_POPULATIONS ? "pop_pull" : (variant == LBWP_KERNEL_TMA ? "tma" : variant == LBWP_KERNEL_MARCH ? "march" : "gather"),
             p->lattice, p->dtype == LBWP_F32 ? "f32" : "f64",
             p->ncomp != 2 ? "" : (variant == LBWP_KERNEL_TMA && !tma2_fused(p)) ? "_c2split" : "_c2");
    rc = load_moments(c, moments, moments_on_device);
    if (rc) return bail(rc);
    *out = c;
    return LBWP_OK;
}

int lbwp_step(lbwp_ctx* c, int64_t n) {
    if (!c || n < 0) return fail(LBWP_EINVAL, "lbwp_step: ctx NULL or n < 0");
    if (n == 0) return LBWP_OK;
    DeviceGuard guard(c->P.device);
    if (!guard.ok) return fail(LBWP_ECUDA, "cudaSetDevice(%d) failed", c->P.device);
    for (int64_t t = 0; t < n; ++t) {
        int rc = c->step_once();
        if (rc) return rc;
    }
    return LBWP_OK;
}

int lbwp_moments(lbwp_ctx* c, void* dst, int dst_on_device) {
    if (!c || !dst) return fail(LBWP_EINVAL, "lbwp_moments: NULL argument");
    DeviceGuard guard(c->P.device);
    if (!guard.ok) return fail(LBWP_ECUDA, "cudaSetDevice(%d) failed", c->P.device);
    void* dev = dst;
    if (!dst_on_device) {
        if (!c->staging) CU(cudaMalloc(&c->staging, dense_bytes(c)));
        dev = c->staging;
    }
    int rc = c->export_dense(dev);
    if (rc) return rc;
    if (!dst_on_device) CU(cudaMemcpyAsync(dst, dev, dense_bytes(c), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    return LBWP_OK;
}

int lbwp_diagnostics(lbwp_ctx* c, double threshold, int nprobes, const int32_t* probe_xyz, lbwp_diag* out, double* probe_rho) {
    if (!c || !out || nprobes < 0 || nprobes > 4096 || (nprobes > 0 && (!probe_xyz || !probe_rho)))
        return fail(LBWP_EINVAL, "lbwp_diagnostics: NULL argument or nprobes outside [0, 4096]");
    for (int p = 0; p < nprobes; ++p)
        if (probe_xyz[3 * p] < 0 || probe_xyz[3 * p] >= c->L.nx || probe_xyz[3 * p + 1] < 0 || probe_xyz[3 * p + 1] >= c->L.ny ||
            probe_xyz[3 * p + 2] < 0 || probe_xyz[3 * p + 2] >= c->L.nz)
            return fail(LBWP_EINVAL, "lbwp_diagnostics: probe %d lies outside the box", p);
    DeviceGuard guard(c->P.device);
    if (!guard.ok) return fail(LBWP_ECUDA, "cudaSetDevice(%d) failed", c->P.device);
    if (!c->staging) CU(cudaMalloc(&c->staging, dense_bytes(c)));
    constexpr int NP = lbwp::DIAG_NSUM + 1;
    const size_t partial_bytes = (size_t)lbwp::DIAG_BLOCKS * NP * sizeof(double), probe_bytes = 4096 * 3 * sizeof(int),
                 out_bytes = (NP + 4096) * sizeof(double);
    if (!c->diag) CU(cudaMalloc(&c->diag, partial_bytes + probe_bytes + out_bytes));
    double* partial = (double*)c->diag;
    int* dprobes = (int*)((char*)c->diag + partial_bytes);
    double* dout = (double*)((char*)c->diag + partial_bytes + probe_bytes);
    int rc = c->export_dense(c->staging);   // the current moments, dense external layout
    if (rc) return rc;
    if (nprobes) CU(cudaMemcpyAsync(dprobes, probe_xyz, (size_t)nprobes * 3 * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    const long long n = (long long)c->L.nx * c->L.ny * c->L.nz;
    if (c->P.dtype == LBWP_F32) {
        if (c->P.ncomp == 1) lbwp::k_diag_partial<float, 1><<<lbwp::DIAG_BLOCKS, lbwp::DIAG_THREADS, 0, c->stream>>>((const float*)c->staging, n, threshold, partial);
        else lbwp::k_diag_partial<float, 2><<<lbwp::DIAG_BLOCKS, lbwp::DIAG_THREADS, 0, c->stream>>>((const float*)c->staging, n, threshold, partial);
        lbwp::k_diag_final<float><<<1, 128, 0, c->stream>>>(partial, lbwp::DIAG_BLOCKS, (const float*)c->staging, c->L.nx, c->L.ny, c->L.nz, dprobes, nprobes, dout);
    } else {
        if (c->P.ncomp == 1) lbwp::k_diag_partial<double, 1><<<lbwp::DIAG_BLOCKS, lbwp::DIAG_THREADS, 0, c->stream>>>((const double*)c->staging, n, threshold, partial);
        else lbwp::k_diag_partial<double, 2><<<lbwp::DIAG_BLOCKS, lbwp::DIAG_THREADS, 0, c->stream>>>((const double*)c->staging, n, threshold, partial);
        lbwp::k_diag_final<double><<<1, 128, 0, c->stream>>>(partial, lbwp::DIAG_BLOCKS, (const double*)c->staging, c->L.nx, c->L.ny, c->L.nz, dprobes, nprobes, dout);
    }
    CU(cudaGetLastError());
    double h[NP + 4096];
    CU(cudaMemcpyAsync(h, dout, (size_t)(NP + nprobes) * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    out->mass[0] = h[0]; out->mass[1] = h[1];
    out->momentum[0] = h[2]; out->momentum[1] = h[3]; out->momentum[2] = h[4];
    out->count_above = (int64_t)(h[6] + 0.5);
    out->rho_mean_above = h[6] > 0.0 ? h[5] / h[6] : 0.0;
    out->rho_max = h[lbwp::DIAG_NSUM];
    for (int p = 0; p < nprobes; ++p) probe_rho[p] = h[NP + p];
    return LBWP_OK;
}

// ---- lbwp_diagnostics_static: the same reduction with no allocation anywhere (include/lbwp.h) ----------------------
// The block partials live in this file-scope device array.  In host code its name is a host-side stand-in, not a device
// address: the address a kernel may use is looked up once per device (that device current) and cached.
static __device__ __align__(256) double g_diag_static_scratch[lbwp::DIAG_BLOCKS * (lbwp::DIAG_NSUM + 1)];
static_assert(sizeof(g_diag_static_scratch) == LBWP_DIAG_STATIC_SCRATCH_BYTES, "include/lbwp.h states the scratch size");
static_assert(LBWP_DIAG_STATIC_NOUT == lbwp::DIAG_NSUM + 1, "include/lbwp.h states the output layout");

namespace {
std::mutex g_diag_static_mu;
double* g_diag_static_addr[LBWP_DIAG_STATIC_MAX_DEVICES] = {};

// `device` is current.  cudaGetSymbolAddress resolves the array in the current device's copy of the module.
int diag_static_scratch(int device, double** ptr) {
    std::lock_guard<std::mutex> lock(g_diag_static_mu);
    if (!g_diag_static_addr[device]) {
        void* p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_diag_static_scratch));
        if (!p) return fail(LBWP_ECUDA, "lbwp_diagnostics_static: cudaGetSymbolAddress returned NULL on device %d", device);
        g_diag_static_addr[device] = (double*)p;
    }
    *ptr = g_diag_static_addr[device];
    return LBWP_OK;
}
}  // namespace

int lbwp_diagnostics_static(int device, int dtype, int ncomp, int nx, int ny, int nz, const void* moments, double threshold,
                            int nprobes, const int32_t* probe_xyz, double* out, void* stream) {
    if (!moments || !out) return fail(LBWP_EINVAL, "lbwp_diagnostics_static: moments or out is NULL");
    if (dtype != LBWP_F32 && dtype != LBWP_F64) return fail(LBWP_EINVAL, "lbwp_diagnostics_static: dtype %d is neither LBWP_F32 nor LBWP_F64", dtype);
    if (ncomp != 1 && ncomp != 2) return fail(LBWP_EINVAL, "lbwp_diagnostics_static: ncomp %d is neither 1 nor 2", ncomp);
    if (device < 0 || device >= LBWP_DIAG_STATIC_MAX_DEVICES)
        return fail(LBWP_EINVAL, "lbwp_diagnostics_static: device %d outside [0, %d)", device, LBWP_DIAG_STATIC_MAX_DEVICES);
    if (nx < 1 || ny < 1 || nz < 1) return fail(LBWP_EINVAL, "lbwp_diagnostics_static: empty box %d x %d x %d", nx, ny, nz);
    if ((double)nx * (double)ny * (double)nz > (double)LBWP_DIAG_STATIC_MAX_NODES)
        return fail(LBWP_EINVAL, "lbwp_diagnostics_static: %d x %d x %d nodes exceed the maximum of %lld (LBWP_DIAG_STATIC_MAX_NODES)",
                    nx, ny, nz, (long long)LBWP_DIAG_STATIC_MAX_NODES);
    if (nprobes < 0 || nprobes > LBWP_DIAG_STATIC_MAX_PROBES)
        return fail(LBWP_EINVAL, "lbwp_diagnostics_static: %d probes outside [0, %d] (LBWP_DIAG_STATIC_MAX_PROBES)", nprobes,
                    LBWP_DIAG_STATIC_MAX_PROBES);
    if (nprobes > 0 && !probe_xyz) return fail(LBWP_EINVAL, "lbwp_diagnostics_static: probe_xyz is NULL with %d probes", nprobes);
    DeviceGuard guard(device);
    if (!guard.ok) return fail(LBWP_ECUDA, "cudaSetDevice(%d) failed", device);
    double* partial = nullptr;
    int rc = diag_static_scratch(device, &partial);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const long long n = (long long)nx * ny * nz;
    const int* probes = (const int*)probe_xyz;
    if (dtype == LBWP_F32) {
        const float* m = (const float*)moments;
        if (ncomp == 1) lbwp::k_diag_partial<float, 1><<<lbwp::DIAG_BLOCKS, lbwp::DIAG_THREADS, 0, st>>>(m, n, threshold, partial);
        else lbwp::k_diag_partial<float, 2><<<lbwp::DIAG_BLOCKS, lbwp::DIAG_THREADS, 0, st>>>(m, n, threshold, partial);
        lbwp::k_diag_final_checked<float><<<1, 128, 0, st>>>(partial, lbwp::DIAG_BLOCKS, m, nx, ny, nz, probes, nprobes, out);
    } else {
        const double* m = (const double*)moments;
        if (ncomp == 1) lbwp::k_diag_partial<double, 1><<<lbwp::DIAG_BLOCKS, lbwp::DIAG_THREADS, 0, st>>>(m, n, threshold, partial);
        else lbwp::k_diag_partial<double, 2><<<lbwp::DIAG_BLOCKS, lbwp::DIAG_THREADS, 0, st>>>(m, n, threshold, partial);
        lbwp::k_diag_final_checked<double><<<1, 128, 0, st>>>(partial, lbwp::DIAG_BLOCKS, m, nx, ny, nz, probes, nprobes, out);
    }
    CU(cudaGetLastError());
    return LBWP_OK;
}

namespace {
int halo_copy(lbwp_ctx* c, int z0, int nplanes, void* packed, bool pack) {
    if (!c || !packed) return fail(LBWP_EINVAL, "lbwp_halo_*: NULL argument");
    if (c->P.scheme != LBWP_MOMENTS) return fail(LBWP_EUNSUPPORTED, "lbwp_halo_*: moments scheme only");
    if (nplanes < 1 || z0 < 0 || z0 + nplanes > c->L.nz) return fail(LBWP_EINVAL, "lbwp_halo_*: planes [%d, %d) leave the box", z0, z0 + nplanes);
    DeviceGuard guard(c->P.device);
    if (!guard.ok) return fail(LBWP_ECUDA, "cudaSetDevice(%d) failed", c->P.device);
    long long field, plane, z0off;
    int nf;
    c->plane_geometry(&field, &plane, &z0off, &nf);
    // nf rows (one per state field) of nplanes contiguous planes each: one strided 2-D copy
    char* state = (char*)c->state_buffer() + (size_t)(z0off + (long long)z0 * plane) * c->esize;
    const size_t width = (size_t)nplanes * plane * c->esize, pitch = (size_t)field * c->esize;
    if (pack) CU(cudaMemcpy2DAsync(packed, width, state, pitch, width, nf, cudaMemcpyDeviceToDevice, c->stream));
    else CU(cudaMemcpy2DAsync(state, pitch, packed, width, width, nf, cudaMemcpyDeviceToDevice, c->stream));
    return LBWP_OK;
}
}  // namespace

size_t lbwp_halo_bytes(const lbwp_ctx* c, int nplanes) {
    if (!c || nplanes < 1 || c->P.scheme != LBWP_MOMENTS) return 0;
    long long field, plane, z0off;
    int nf;
    c->plane_geometry(&field, &plane, &z0off, &nf);
    return (size_t)nf * nplanes * plane * c->esize;
}
int lbwp_halo_pack(lbwp_ctx* c, int z0, int nplanes, void* dst) { return halo_copy(c, z0, nplanes, dst, true); }
int lbwp_halo_unpack(lbwp_ctx* c, int z0, int nplanes, const void* src) { return halo_copy(c, z0, nplanes, const_cast<void*>(src), false); }

int lbwp_set_moments(lbwp_ctx* c, const void* moments, int on_device) {
    if (!c) return fail(LBWP_EINVAL, "ctx is NULL");
    DeviceGuard guard(c->P.device);
    if (!guard.ok) return fail(LBWP_ECUDA, "cudaSetDevice(%d) failed", c->P.device);
    return load_moments(c, moments, on_device);
}

int64_t lbwp_steps_done(const lbwp_ctx* c) { return c ? c->steps : -1; }
int lbwp_launches_per_step(const lbwp_ctx* c) { return c ? c->launches_per_step : 0; }
const char* lbwp_kernel_name(const lbwp_ctx* c) { return c ? c->name : ""; }

int lbwp_sync(lbwp_ctx* c) {
    if (!c) return fail(LBWP_EINVAL, "ctx is NULL");
    DeviceGuard guard(c->P.device);
    CU(cudaStreamSynchronize(c->stream));
    return LBWP_OK;
}

int lbwp_destroy(lbwp_ctx* c) {
    if (!c) return LBWP_OK;
    DeviceGuard guard(c->P.device);
    cudaStreamSynchronize(c->stream);
    if (c->owns)
        for (int k = 0; k < 2; ++k)
            if (c->buf[k]) cudaFree(c->buf[k]);
    if (c->grad) cudaFree(c->grad);
    if (c->staging) cudaFree(c->staging);
    if (c->diag) cudaFree(c->diag);
    delete c;
    return LBWP_OK;
}

const char* lbwp_last_error(void) { return g_err; }

}  // extern "C"
