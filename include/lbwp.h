/*
 * lbwp.h -- C ABI of the B200 (sm_100a) "lattice Boltzmann without populations" library.
 *
 * Method: arxiv 2301.01622 ("Lightweight Lattice Boltzmann").  Citations are
 * PAPER.md:<line> (+ equation); "Cn" are the readings listed in DESIGN.md.
 *
 * One context = one periodic box on one GPU.  The state of the scheme is the set
 * of hydrodynamic moments per node, H = [rho, u_a, P_ab] (Eq. 1-3),
 * kept in two ping-pong device buffers ("Flip-Flop").  lbwp_step()
 * advances it by the fused Reconstruct-Collide-Stream-Project update
 * (Eq. 8 at the neighbour, Eq. 9 pull, Eq. 1-3 at the node).
 *
 * External moment layout (input of lbwp_init, output of lbwp_moments): dense SoA
 * [M][nz][ny][nx], x fastest, element type = params.dtype.
 *   ncomp == 1, M = 10: rho, ux, uy, uz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz
 *   ncomp == 2, M = 11: rhoA, rhoB, ux, uy, uz, Pxx, Pyy, Pzz, Pxy, Pxz, Pyz
 * P is the full second moment sum_i f_i c_ia c_ib (Eq. 3), u is the
 * velocity, both of the total fluid for ncomp == 2.
 * The internal device layout (ghost layers, row padding, deviation storage) is
 * private to the library and not visible through this interface.
 *
 * Every function returns LBWP_OK (0) or a negative lbwp_status; nothing throws or
 * aborts.  lbwp_last_error() gives the text of the calling thread's last failure.
 * There is no CPU fallback: without a CUDA device of compute capability 10.x
 * lbwp_init fails with LBWP_EUNSUPPORTED / LBWP_ECUDA.
 */
#ifndef LBWP_H
#define LBWP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lbwp_ctx lbwp_ctx; /* opaque; owned by the library */

enum lbwp_status {
    LBWP_OK = 0,
    LBWP_EINVAL = -1,      /* bad argument (lattice, dtype, ncomp, sizes, tau, NULL) */
    LBWP_ENOMEM = -2,      /* device or host allocation failed */
    LBWP_ECUDA = -3,       /* a CUDA runtime call failed; see lbwp_last_error() */
    LBWP_EUNSUPPORTED = -4 /* device is not sm_100, or the combination is not built */
};
enum lbwp_dtype { LBWP_F32 = 0, LBWP_F64 = 1 };
enum lbwp_scheme {
    LBWP_MOMENTS = 0,    /* the paper's scheme: moments only */
    LBWP_POPULATIONS = 1 /* comparison point: population-storing pull BGK */
};
enum lbwp_kernel {
    LBWP_KERNEL_AUTO = 0,   /* fastest kernel built for the combination */
    LBWP_KERNEL_GATHER = 1, /* one thread per node, 27/19-neighbour gather through L1/L2 */
    LBWP_KERNEL_MARCH = 2,  /* shared-memory tiles, z-marching register accumulators (any box size) */
    LBWP_KERNEL_TMA_SPLIT = 4, /* two-component only: collide pass + TMA stencil pass (the paper's split form),
                               kept for comparison with the fused form LBWP_KERNEL_TMA uses */
    LBWP_KERNEL_TMA = 3     /* TMA-fed stencil on the collided ("S-form") moments, collision as epilogue:
                               D3Q27 and D3Q19, nx a multiple of 64 (fp32) / 32 (fp64), ny of 8; one launch per step,
                               two-component runs included (gradient, perturbation and recolouring fused in) */
};

typedef struct lbwp_params {
    int32_t struct_size; /* = sizeof(lbwp_params); ABI check */
    int32_t lattice;     /* 19 | 27  (D3Q19 is the paper's; D3Q27 reading C10) */
    int32_t dtype;       /* lbwp_dtype: precision of the stored state AND of the arithmetic */
    int32_t ncomp;       /* 1 | 2 (2 = colour-gradient two-component; reading C6) */
    int32_t scheme;      /* lbwp_scheme */
    int32_t kernel;      /* lbwp_kernel; AUTO unless a test wants a specific one */
    int32_t nx, ny, nz;  /* periodic box (reading C13), each >= 1 */
    int32_t device;      /* CUDA device ordinal */
    double tau;          /* relaxation time > 0.5; omega = 1/tau, nu = cs^2 (tau - 1/2) (C3) */
    double A;            /* ncomp == 2: perturbation (surface tension) strength; else ignored */
    double beta;         /* ncomp == 2: recolouring strength; else ignored */
    void *stream;        /* cudaStream_t all work is enqueued on; NULL = legacy default stream */
    void *buf[2];        /* optional caller-owned DEVICE buffers, each >= lbwp_state_bytes() bytes and
                            256-byte aligned (e.g. a torch tensor's data_ptr); must outlive the ctx.
                            NULL, NULL => the library allocates and frees them. */
    double A_h;          /* ncomp == 2, moments scheme: strength of the near-contact repulsion
                            F_rep = -A_h[h(x)] n delta_I (Eq. 10; readings C20-C24 of DESIGN.md:
                            delta_I = |grad phi|/2, n the outward normal, A_h[h] = A_h for h <= h_c and 0 beyond,
                            Guo forcing).  0 = off (BASELINE's configs).  Non-zero adds two launches per step behind
                            the fused two-component TMA kernel (min / max of rA per box of nodes, then a pass over
                            the boxes that hold an interface: it finds the facing interfaces and applies the forcing
                            to the collided moments in place), or, for boxes the TMA tiles do not divide and with
                            LBWP_KERNEL_GATHER, selects the generic kernel (three launches per step: gradient,
                            contact search, step); LBWP_EUNSUPPORTED with LBWP_KERNEL_TMA_SPLIT / MARCH.  The force
                            looks floor(h_c) + 1 planes beyond a node: slabs then need H = floor(h_c) + 3 halo planes. */
    double h_c;          /* cut-off distance of the near-contact force in lattice units (> 0 when A_h != 0) */
} lbwp_params;

/* Bytes of ONE internal state buffer (ghost layers and padding included) for these
 * params; 0 if they are invalid.  Host-only, no CUDA call. */
size_t lbwp_state_bytes(const lbwp_params *params);

/* Number of moment fields M of the external layout (10 or 11); 0 if invalid. */
int lbwp_num_moments(const lbwp_params *params);

/* Create a context and load the initial moments (external layout above; `moments`
 * is a HOST pointer if moments_on_device == 0, else a DEVICE pointer on
 * params->device).  For scheme == LBWP_POPULATIONS the initial populations are the
 * Eq. 4 reconstruction of these moments; with ncomp == 2 one set
 * per colour, split as f^A = (rho_A / rho) f.  Synchronises the stream
 * before returning.  *out is set only on success. */
int lbwp_init(const lbwp_params *params, const void *moments, int moments_on_device, lbwp_ctx **out);

/* Enqueue n >= 0 time steps on the context's stream; asynchronous (no sync).  One step = for every node x and
 * direction c_i: Eq. 8 at x - c_i, pulled to x (Eq. 9), summed into the new moments
 * (Eq. 1-3); ncomp == 2: with the colour-gradient perturbation and recolouring (C6).
 * n == 0 is a no-op.  Launch errors are reported; execution errors surface at the
 * next synchronising call. */
int lbwp_step(lbwp_ctx *ctx, int64_t n);

/* Write the current moments H = [rho, u_a, P_ab], i.e. the POST-STREAM, PRE-COLLISION moments of
 * Eq. 1-3 at the current time (reading C5: Eq. 8-9 collide at the neighbour, then stream), external layout,
 * M*nz*ny*nx elements of params.dtype,
 * to `dst` (HOST pointer if dst_on_device == 0, else DEVICE pointer).  Synchronises
 * the stream.  Does not change the state. */
int lbwp_moments(lbwp_ctx *ctx, void *dst, int dst_on_device);

/* The paper's run-time diagnostics of the CURRENT state (Fig. 2, 3, 5, 7), one fused reduction
 * in fp64 over all nodes.  "Density" is the density of the first component (the droplet fluid, whose field ranges
 * from 0 to 1): rhoA for ncomp == 2, rho for ncomp == 1.
 *   mass[2]      sum over nodes of rhoA and of rhoB (0 for ncomp == 1)              (Eq. 1 summed over the box)
 *   momentum[3]  sum over nodes of rho u, rho = rhoA + rhoB                          (Eq. 2 summed over the box)
 *   rho_mean_above, count_above   <density>_{density > threshold} and the number of such nodes (the paper's
 *                <rho>_{rho > 0.5}; mean is 0 if no node qualifies)
 *   rho_max      maximum of the density (the paper's rho_N,MAX)
 * probe_xyz: nprobes triples (x, y, z) of node coordinates (HOST pointer, may be NULL if nprobes == 0);
 * probe_rho: the density at those nodes (HOST pointer).  Synchronises the stream; does not change the state.
 * LBWP_EINVAL for a NULL argument, nprobes < 0 or a probe outside the box. */
typedef struct lbwp_diag {
    double mass[2];
    double momentum[3];
    double rho_mean_above;
    double rho_max;
    int64_t count_above;
} lbwp_diag;
int lbwp_diagnostics(lbwp_ctx *ctx, double threshold, int nprobes, const int32_t *probe_xyz, lbwp_diag *out,
                     double *probe_rho);

/* The same reduction for callers that may not allocate: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc.  This entry point calls no cudaMalloc / cudaFree / allocating
 * library routine, needs no context, enqueues two kernels on `stream` and returns without synchronising.  Its only
 * scratch (the 592 block partials of 9 doubles: LBWP_DIAG_STATIC_SCRATCH_BYTES) is a file-scope device array of the
 * library, held by every GPU that loads the library until the process exits.
 *   device     CUDA device ordinal in [0, LBWP_DIAG_STATIC_MAX_DEVICES) that holds every pointer below
 *   dtype, ncomp, nx, ny, nz   as in lbwp_params; nx*ny*nz <= LBWP_DIAG_STATIC_MAX_NODES
 *   moments    DEVICE pointer, the dense external layout of lbwp_moments: [M][nz][ny][nx], M = lbwp_num_moments(ncomp)
 *   probe_xyz  DEVICE pointer, nprobes <= LBWP_DIAG_STATIC_MAX_PROBES triples (x, y, z); may be NULL if nprobes == 0
 *   out        DEVICE pointer, LBWP_DIAG_STATIC_NOUT + nprobes doubles, all written by the call:
 *              [0] sum rhoA  [1] sum rhoB  [2..4] sum rho u  [5] sum of the density over the nodes above the threshold
 *              [6] number of those nodes  [7] 0  [8] maximum density  [9 + p] density at probe p (NaN if the probe
 *              lies outside the box: the coordinates are device data the host cannot check)
 *   stream     cudaStream_t (NULL: the default stream)
 * Sums are added in the same order as lbwp_diagnostics adds them, so [0..8] equal its results bit for bit
 * (rho_mean_above = out[5] / out[6]).
 * The scratch is SHARED by every call on a device and keeps the last call's contents.  Nothing in it has to start at
 * zero (the first kernel writes every element the second reads), but two calls that overlap on the GPU (different
 * streams without an ordering between them, or concurrent branches of one graph) race on it: order them.
 * The first call on each device resolves the array's device address (cudaGetSymbolAddress, which may load the
 * library's module): make one call per device before starting a stream capture.
 * LBWP_EINVAL for a NULL pointer, a bad dtype / ncomp / device, or a size beyond the maxima above (the text from
 * lbwp_last_error names the limit); LBWP_ECUDA if the address lookup or a launch fails. */
#define LBWP_DIAG_STATIC_SCRATCH_BYTES 42624 /* 592 blocks x 9 doubles */
#define LBWP_DIAG_STATIC_MAX_NODES 2147483648LL /* 2^31, the library's own grid limit */
#define LBWP_DIAG_STATIC_MAX_PROBES 4096
#define LBWP_DIAG_STATIC_MAX_DEVICES 64
#define LBWP_DIAG_STATIC_NOUT 9
int lbwp_diagnostics_static(int device, int dtype, int ncomp, int nx, int ny, int nz, const void *moments,
                            double threshold, int nprobes, const int32_t *probe_xyz, double *out, void *stream);

/* z-slab decomposition over several GPUs (the paper's motivation are grids of billions of nodes,
 * PAPER.md:163-167).  A rank's context is an ordinary periodic box whose first and last H planes are HALO planes:
 * copies of the neighbouring ranks' boundary planes (H = 1; H = 2 for ncomp == 2 moments, whose colour gradient
 * reaches two planes; H = floor(h_c) + 3 with the near-contact force, whose interface walk and the gradients on its
 * way reach floor(h_c) + 1 planes beyond the two the step leaves wrong).
 * One step of the decomposed box = lbwp_step(ctx, 1) on every rank, then every rank packs its
 * H lowest and H highest OWNED planes of the new state, sends them to its z neighbours (NCCL send/recv, or a peer
 * copy) and unpacks what it receives into its halo planes.  The planes the step computed INTO the halo are garbage
 * (the box wrapped onto itself there) and are overwritten by the unpack.  The packed format is the library's private
 * state layout: only contexts with identical params and step count may exchange it.
 *   lbwp_halo_bytes   bytes of nplanes packed planes (0 on error)
 *   lbwp_halo_pack    planes [z0, z0 + nplanes) of the CURRENT state -> dst (DEVICE pointer), asynchronous on the stream
 *   lbwp_halo_unpack  src (DEVICE pointer) -> planes [z0, z0 + nplanes) of the current state, asynchronous
 * LBWP_EINVAL if the plane range leaves the box. */
size_t lbwp_halo_bytes(const lbwp_ctx *ctx, int nplanes);
int lbwp_halo_pack(lbwp_ctx *ctx, int z0, int nplanes, void *dst);
int lbwp_halo_unpack(lbwp_ctx *ctx, int z0, int nplanes, const void *src);

/* Replace the state by new moments (same conventions as lbwp_init); step counter -> 0. */
int lbwp_set_moments(lbwp_ctx *ctx, const void *moments, int moments_on_device);

/* Time steps taken since init / set_moments. */
int64_t lbwp_steps_done(const lbwp_ctx *ctx);

/* Number of kernel launches lbwp_step enqueues per time step for this context
 * (1 for the fused single-component kernels). */
int lbwp_launches_per_step(const lbwp_ctx *ctx);

/* Name of the step kernel variant in use ("march27_f32", "gather19_f64_c2", ...);
 * static storage, never freed by the caller. */
const char *lbwp_kernel_name(const lbwp_ctx *ctx);

/* Synchronise the context's stream. */
int lbwp_sync(lbwp_ctx *ctx);

/* Free the context and every buffer the library allocated (never the caller's buf[]). */
int lbwp_destroy(lbwp_ctx *ctx);

/* Text of the calling thread's last error ("" if none); thread-local static storage. */
const char *lbwp_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LBWP_H */
