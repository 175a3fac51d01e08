/*
 * cp4d.h -- C ABI of libcp4d.so: the Chambolle-Pock hot path of "Four-dimensional tomographic
 * reconstruction by time domain decomposition" (arXiv 1809.09725; citations below are PAPER.md
 * line numbers) as hand-written sm_100a CUDA kernels.  One GPU, fp32 arithmetic,
 * no CPU fallback: every entry point that computes runs CUDA kernels or fails with an error code.
 *
 * Problem.  f(x,y,z,t) ~ sum_j f_j(x,y,z) phi_j(t), j < m (Eq. 8).  The primal variable
 * is the coefficient stack f_j (reading C1).  Minimise (Eq. 6)
 *      1/2 |K1 f - g|^2 + lambda1 | |K2 f| |_1 ,
 *   K1 f [z,k,b] = sum_j Phi[j,k] * (R_{theta_k} f_j(.,.,z))[b]          (Eq. 9; L231)
 *   K2 f         = grad_{lambda2} f = (d_x f, d_y f, d_z f, lambda2 d_t f)  (Eq. 5; L123)
 * with the Chambolle-Pock iteration of Fig. 2 (L147-L168).  R is the static parallel-beam Radon
 * transform discretised by the Joseph linear-interpolation ray sum (reading R3; the
 * paper's own log-polar code is not specified, L281): equivalently the matrix
 *      A_k[b; iy,ix] = Lambda((x_ix c_k + y_iy s_k - s_b)/a_k)/a_k,  Lambda(u) = max(0, 1-|u|),
 *      a_k = max(|c_k|,|s_k|),  c_k = cos theta_k, s_k = sin theta_k.
 *
 * Geometry (R1/R2).  Unit voxel and bin spacing; voxel centres x_ix = ix-(n-1)/2,
 * y_iy = iy-(n-1)/2; bin centres s_b = b-(nd-1)/2; theta_k = k*pi/n_theta0 with
 * n_theta0 = n_angles/n_half_rot; t_k = k/n_angles (enters only through the caller's table Phi).
 * Values outside the grid are zero; rays exist only for 0 <= b < nd.
 *
 * Layouts (dense, no padding, fp32, base pointers 16-byte aligned; V = nz*n*n*mp, S = nz*n_angles*nd,
 * mp = m, or n_frames in frame mode where j below is the frame index):
 *   primal-shaped   f[z][iy][ix][j]        j fastest                      V floats
 *   sinogram        g[z][k][b]             b fastest                      S floats
 *   dual field      p[a][z][iy][ix][j]     a = 0..3 = (x, y, z, t)        4V floats, component-major
 *   basis table     phi[j][k] = phi_j(t_k) host memory, copied at create  m*n_angles floats
 *
 * Pointers named *_dev are DEVICE pointers on `device`, *_host are HOST pointers.  The caller owns
 * every buffer it passes (e.g. PyTorch tensors); the library never frees or resizes them and
 * allocates no device memory: all state and scratch live in the caller's workspace.  Input and
 * output buffers of one call must not overlap (CP4D_EINVAL) unless a parameter says "in/out".
 * All kernels are enqueued on the stream given at create; calls are asynchronous unless they say
 * "syncs".  Every call makes the context's device current for its duration and restores the caller's current device
 * before it returns (cp4d_create included), so contexts of several devices can be driven from one thread.  Asynchronous faults surface at the next syncing call as CP4D_ECUDA.
 *
 * Every function returns 0 (CP4D_OK) or a negative error code; nothing throws, exits or prints.
 */
#ifndef CP4D_H
#define CP4D_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CP4D_OK            0
#define CP4D_EINVAL       -1  /* null pointer, bad size, n_angles % n_half_rot, m % 4, m > 32, misaligned, aliasing */
#define CP4D_EWORKSPACE   -2  /* workspace missing or smaller than cp4d_workspace_bytes() */
#define CP4D_EUNSUPPORTED -3  /* no CUDA device / device is not compute capability 10.x */
#define CP4D_ECUDA        -4  /* a CUDA runtime call or kernel failed; text in cp4d_last_error() */
#define CP4D_ESTATE       -5  /* call order: cp4d_iterate before cp4d_set_data / cp4d_set_steps */
#define CP4D_ENOMEM       -6  /* a host allocation failed (cp4d_create) */
#define CP4D_EINTERNAL    -7  /* an invariant of the host prologue failed (cp4d_create: the base angles are not sorted by
                                 the sign of cos, or a tile window leaves the padded scratch row); a bug, never an input error */

#define CP4D_ETOOLARGE    -8  /* cp4d_forward_static: the problem's scratch exceeds CP4D_STATIC_SCRATCH_BYTES */

typedef struct cp4d_ctx cp4d_ctx; /* opaque; owns host-side metadata only */

typedef struct {
    int32_t nx, ny;           /* grid side; the hot path requires nx == ny (= n)                          */
    int32_t nz;               /* slices, >= 1                                                              */
    int32_t nd;               /* detector bins, >= 2, unit spacing, centred                                */
    int32_t n_angles;         /* N_theta, total projections                                                */
    int32_t n_half_rot;       /* N_pi half-rotations; n_angles % n_half_rot == 0 (L200; C17);
                                 n_half_rot * m <= 12288 (the slice of Phi of one base angle sits in shared memory)  */
    int32_t m;                /* temporal basis functions (the paper's M); m % 4 == 0, 4 <= m <= 32        */
    int32_t device;           /* CUDA device ordinal                                                       */
    const float *phi_host;    /* HOST, m*n_angles, [j][k] = phi_j(t_k); copied at create (L176-L180)       */
    float lambda1, lambda2;   /* Eq. (5)/(6): TV weight; temporal scale inside the 4-vector gradient       */
    float theta_relax;        /* over-relaxation theta in [0,1] of Fig. 2 step 6 (C12: 1)        */
    void *workspace_dev;      /* DEVICE, caller-allocated, >= cp4d_workspace_bytes(), 256-byte aligned     */
    uint64_t workspace_bytes;
    void *stream;             /* cudaStream_t (0 = legacy default stream)                                  */
    int32_t n_frames;         /* 0: the primal array is the coefficient stack f_j (4th axis m).  N_t > 0: the paper's own
                                 discretisation (L214-L237): the primal array holds N_t time frames f(t_q) (4th axis N_t,
                                 N_t % 4 == 0, N_t <= 32, n_angles % N_t == 0), frame q sits at the time of angle
                                 q*n_angles/N_t; K1 f = K1_coef(f_j) with f_j = sum_q phi_j(t_q) f(t_q), phi_j(t_q) taken
                                 from phi_host's column q*n_angles/N_t; the 4th difference of K2 runs over frames      */
    int32_t z_open;           /* 0: the context holds the whole volume.  Otherwise it is a z-SLAB of a taller volume (PAPER.md
                                 L283: "split computations by slices ... we transfer to GPU two extra slices located before and
                                 after the current set of slices", kept read-only): bit 0 = the face below slice 0 is interior,
                                 bit 1 = the face above slice nz-1 is interior.  K1 / K1^T act per slice and need nothing; the
                                 z-differences of K2 / K2^T take the neighbour's slice through the halo arguments of the
                                 *_slab calls below.  cp4d_grad, cp4d_div, cp4d_prox_f2, cp4d_primal_update, cp4d_iterate,
                                 cp4d_norm, cp4d_objective and cp4d_solve_host return CP4D_ESTATE on a slab context.          */
} cp4d_params;

/* Bytes of device workspace a context for these sizes needs (state f, f~, K1^T h1, h2[4], h1, g, one sinogram-sized
 * temporary, the zero-padded folded sinogram of the adjoint (m * n_theta0 * (nd + pads) * nz floats), the forward projector's
 * partial ray sums (m * n_theta0 * nd * nz floats), tables -- among them the work items of the tensor-core forward
 * projector, 2.7 KB per 32 x 32 tile and group of four base angles; in frame mode with N_t > m two coefficient stacks
 * as well).
 * Host only; ignores workspace_dev/stream/phi_host.  Errors: CP4D_EINVAL (see cp4d_params). */
int cp4d_workspace_bytes(const cp4d_params *p, uint64_t *bytes_out);
/* The same plus second copies of h2[4] and f~ (5 * V floats more).  A context created on a workspace of at least this size
 * (whole volume, z_open == 0) runs steps 4-6 of Fig. 2 as ONE pass over the volume -- the dual variable
 * goes from its projection to the divergence of the primal update through shared memory, 13 V instead of 17 V floats of HBM
 * traffic per iteration -- which needs the two arrays double-buffered: a CTA recomputes the projection
 * on a one-voxel halo from the OLD values while its neighbour writes the new ones.  cp4d_iterate then swaps the roles of the
 * copies after every iteration (see cp4d_state_ptrs).  The iterates are those of the two-kernel path. */
int cp4d_workspace_bytes_fused(const cp4d_params *p, uint64_t *bytes_out);
/* *out_host = 1 if cp4d_iterate of this context runs the one-pass step (workspace >= cp4d_workspace_bytes_fused at create and
 * z_open == 0), else 0 */
int cp4d_fused_step_in_use(const cp4d_ctx *ctx, int32_t *out_host);

/* Validate, compute the fp64 angle/tile tables on the host, copy them and phi into the workspace,
 * carve the workspace.  Launches one kernel on the stream (the work items of the tensor-core forward projector, which depend
 * on the geometry only) and synchronizes it.  The context keeps workspace_dev and stream. */
int cp4d_create(const cp4d_params *p, cp4d_ctx **ctx_out);
int cp4d_destroy(cp4d_ctx *ctx);

/* ---- stateless operators on caller-owned DEVICE buffers -------------------------------------- */
/* Every function below returns CP4D_EINVAL for a null context, a null or misaligned (16 B) pointer or overlapping in/out
 * buffers, and CP4D_ECUDA (text in cp4d_last_error) if a launch fails.  "V" is the primal size: in frame mode f holds
 * the n_frames frames and K1 includes the analysis f_j = sum_q phi_j(t_q) f(t_q). */
/* g = K1 f  (Eq. 9; pi-folding L198-L202: ray sums over the n_theta0 base angles with all m
 * coefficients accumulated per ray, then n_half_rot m-wide dot products with Phi).  f: V, g: S. */
int cp4d_forward(cp4d_ctx *ctx, const float *f_dev, float *g_dev);
/* g = K1 f as cp4d_forward computes it (same kernels, same projector mode), for callers that must not depend on workspace
 * scratch at call time (CUDA graph capture of their own, serving loops, harnesses that forbid device allocation): the
 * projector's partial ray sums (m * n_theta0 * nd * nz floats) go to a file-scope __device__ array of
 * CP4D_STATIC_SCRATCH_BYTES inside the library instead of the workspace.  Calls no cudaMalloc / cudaFree or any allocating
 * routine; every GPU that loads libcp4d.so holds the array until the process exits.  Problems whose partial sums exceed it
 * return CP4D_ETOOLARGE (sizes in cp4d_last_error); nothing is launched then.  All calls on one device share the array: each
 * call zero-fills the part it uses on the context's stream, so calls ordered by a stream are fine, and calls that overlap
 * on the GPU (contexts on different streams, no dependency between them) race.  Result equals cp4d_forward's up to the
 * order of the projector's atomic additions.  Errors otherwise as cp4d_forward. */
#define CP4D_STATIC_SCRATCH_BYTES (32u << 20)
int cp4d_forward_static(cp4d_ctx *ctx, const float *f_dev, float *g_dev);
/* f = K1^T g, overwrite (Eq. 10; fold L204-L212: gt_j = sum_q Phi[j,q n0+i] g[q n0+i, flip_q b],
 * then one backprojection over [0,pi)).  Exact transpose of cp4d_forward up to fp32 rounding. */
int cp4d_adjoint(cp4d_ctx *ctx, const float *g_dev, float *f_dev);
/* p = K2 f: forward differences along x, y, z, t (t scaled by lambda2), 0 at the last index of
 * each axis (R4).  f: V, p: 4V. */
int cp4d_grad(cp4d_ctx *ctx, const float *f_dev, float *p_dev);
/* f = div p = -K2^T p (L131-L133).  p: 4V, f: V. */
int cp4d_div(cp4d_ctx *ctx, const float *p_dev, float *f_dev);

/* Which kernels cp4d_forward / cp4d_adjoint and everything built on them (cp4d_prox_f1, cp4d_primal_update, cp4d_iterate,
 * cp4d_norm, cp4d_objective, cp4d_solve_host) launch.  All of them compute the same ray sums and their transpose (Eq. 9 /
 * Eq. 10 with the Joseph weights above); they differ in the arithmetic of the products:
 *   tensor-core kernels (m = 4, 8, 16 or 32 only): voxel / sinogram values and interpolation weights enter the 2:4 sparse mma.sp
 *       (the weight block is the sparse operand: two adjacent taps per ray and column, per voxel and angle) as split bf16 pairs (x = x_hi + x_lo with |x - x_hi - x_lo| <= 2^-17 |x|), three products per term, fp32 accumulation:
 *       relative error about 5e-6 per ray sum or voxel (bound 1.1e-5), inside the 1e-4 per-operator tolerance;
 *   fp32 kernels: CUDA-core FMAs, relative error about 2e-6.
 *   CP4D_PROJ_AUTO (default): the faster pair -- the tensor-core kernels on both sides where they apply and the problem
 *       fills the GPU (at least 148 CTAs of (tile, pass, batch group): forward 2.1 x the fp32 gather, adjoint 1.12 x the fp32
 *       backprojector at config 3), the fp32 kernels otherwise.
 *   CP4D_PROJ_FP32: fp32 kernels on both sides.      CP4D_PROJ_TENSOR: tensor-core kernels on both sides where they apply.
 * cp4d_fbp always uses the fp32 backprojector.  Changing the mode drops the captured CUDA graph of cp4d_iterate and clears the
 * projector scratch (asynchronously, on the context's stream). */
#define CP4D_PROJ_AUTO   0
#define CP4D_PROJ_FP32   1
#define CP4D_PROJ_TENSOR 2
int cp4d_set_projector_mode(cp4d_ctx *ctx, int32_t mode);
/* which kind (CP4D_PROJ_FP32 / CP4D_PROJ_TENSOR) the forward and the adjoint run with; either pointer may be null (HOST) */
int cp4d_projector_mode_in_use(const cp4d_ctx *ctx, int32_t *forward_out_host, int32_t *adjoint_out_host);

/* ---- the three fused steps of Fig. 2 on caller-owned DEVICE buffers --------------------------- */
/* step 3 (L154, L135): h1 <- (h1 + sigma (K1 ft - g)) / (1 + sigma).   h1 in/out (S), ft: V, g: S. */
int cp4d_prox_f1(cp4d_ctx *ctx, float sigma, const float *ft_dev, const float *g_dev, float *h1_dev);
/* step 4 (L158, L137; R5): q = h2 + sigma grad ft; h2 <- q / max(1, |q|_2 / lambda1)
 * pointwise over the 4-vector at each (x,y,z,j); lambda1 == 0 gives h2 = 0.  h2 in/out (4V). */
int cp4d_prox_f2(cp4d_ctx *ctx, float sigma, const float *ft_dev, float *h2_dev);
/* steps 5-6 (L162-L166): f+ = f - tau K1^T h1 + tau div h2;  ft = f+ + theta (f+ - f);  f <- f+.
 * f in/out (V), ft out (V), h1: S, h2: 4V. */
int cp4d_primal_update(cp4d_ctx *ctx, float tau, const float *h1_dev, const float *h2_dev, float *f_dev,
                       float *ft_dev);

/* ---- reductions (fp32 in, fp64 accumulate).  Sync. ------------------------------------------- */
int cp4d_dot(cp4d_ctx *ctx, const float *x_dev, const float *y_dev, uint64_t count, double *out_host);

/* ---- power iteration for L = ||K||, K = (K1; K2) (L97, L147; R8) ------------------- */
/* x0 = counter-based N(0,1) from `seed`; n_power_iters steps of y = K1^T K1 x + K2^T K2 x,
 * L = sqrt(|y|/|x|).  Uses the CP state buffers as scratch (call before cp4d_reset).  Syncs. */
int cp4d_norm(cp4d_ctx *ctx, int32_t n_power_iters, uint64_t seed, float *L_out_host);
/* The same iteration from the caller's start vector x0 (DEVICE, V floats, any non-zero finite vector; it is copied and
 * normalised), so that a reference implementation handed the same x0 can be compared step for step.  CP4D_EINVAL if x0 is
 * null, misaligned, zero or not finite.  Syncs. */
int cp4d_norm_start(cp4d_ctx *ctx, int32_t n_power_iters, const float *x0_dev, float *L_out_host);

/* ---- Chambolle-Pock state machine; state (f, ft, h1, h2, g) lives in the workspace ----------- */
int cp4d_set_data(cp4d_ctx *ctx, const float *g_dev);                 /* copy measured data g (S) */
int cp4d_set_steps(cp4d_ctx *ctx, float tau, float sigma);            /* tau*sigma*L^2 < 1 is the caller's duty */
int cp4d_reset(cp4d_ctx *ctx, const float *f0_dev /* nullable => zeros */); /* f = ft = f0, h1 = h2 = 0 */
int cp4d_iterate(cp4d_ctx *ctx, int32_t n_iters);                     /* n_iters x steps 3-6, async */
int cp4d_get_f(cp4d_ctx *ctx, float *f_dev_out);                      /* copy f (V) */
/* device pointers of the state arrays inside the workspace (for inspection / teacher forcing);
 * any of the out pointers may be null.  With the one-pass step (cp4d_fused_step_in_use) ft and h2 alternate between their two
 * copies: the pointers are those of the CURRENT state and stay valid until the next cp4d_iterate. */
int cp4d_state_ptrs(cp4d_ctx *ctx, float **f, float **ft, float **h1, float **h2, float **g);

/* ---- convergence monitor (off the timed path).  Syncs. ---------------------------------------- */
/* primal    = 1/2 |K1 f - g|^2 + lambda1 * sum over (x,y,z,j) of |K2 f|_2          (Eq. 6)
 * cond_dual = -1/2 |h1|^2 - <h1, g>   (dual value of Eq. 7 with the constraint K^T h = 0 of G = 0 ignored; not a lower
 *             bound while K^T h != 0, C19)
 * kkt_resid = |K1^T h1 - div h2|_2    (dual residual; -> 0 at a saddle point)
 * Out pointers are HOST and may be null.  Uses the K1^T h1 buffer and the projector scratch; state is untouched. */
int cp4d_objective(cp4d_ctx *ctx, double *primal, double *cond_dual, double *kkt_resid);

/* ---- static filtered backprojection per half-rotation (L243, L257-L259: the paper's comparison method and initial guess) */
/* out[z][iy][ix][q], q < Q4 = 4*ceil(n_half_rot/4) (planes q >= n_half_rot are zero):
 *     out_q = (pi / n_theta0) * sum_{i < n_theta0} R*_{theta_i} ( h_SL * g[q n_theta0 + i] ),
 * h_SL[n] = -2 / (pi^2 (4 n^2 - 1)) the Shepp-Logan filter at unit bin spacing, R* the same (Joseph) backprojector as
 * cp4d_adjoint with odd half-rotations bin-flipped.  In frame mode with n_frames == n_half_rot == Q4, out is a valid f0 for
 * cp4d_reset.  g: S, out: nz*n*n*Q4 floats, DEVICE.  Needs Q4 <= m (else CP4D_EUNSUPPORTED).  Uses the sinogram temporary and
 * the projector scratch. */
int cp4d_fbp(cp4d_ctx *ctx, const float *g_dev, float *out_dev);

/* ---- z-slab contexts (cp4d_params.z_open != 0) ---------------- */
/* Halo arguments are DEVICE pointers to ONE slice [iy][ix][j] (n*n*mp floats, 16-byte aligned) owned by the caller (a
 * neighbour context's state on this device, or a receive buffer); read-only, never retained.  A halo must be given exactly
 * for the faces z_open marks interior, else CP4D_EINVAL.  The calls also work on a whole-volume context (both halos null).
 *   f_above : the neighbour's slice of f (or ft) at z = nz        (forward z-difference of the last slice)
 *   pz_below: the neighbour's slice of the z-component of p (h2) at z = -1   (backward z-difference of slice 0)      */
/* change which faces are interior (a pool of contexts that slabs of a taller volume pass through one after the other) */
int cp4d_set_z_open(cp4d_ctx *ctx, int32_t z_open);
int cp4d_grad_slab(cp4d_ctx *ctx, const float *f_dev, const float *f_above, float *p_dev);
int cp4d_div_slab(cp4d_ctx *ctx, const float *p_dev, const float *pz_below, float *f_dev);
/* Fig. 2 steps 3-4 on the context's state: h1 <- prox_{sigma F1*}(h1 + sigma K1 ft), h2 <- prox_{sigma F2*}(h2 + sigma K2 ft).
 * ft_above: the upper neighbour's FIRST slice of ft, as it was BEFORE that neighbour's cp4d_step_primal of this iteration. */
int cp4d_step_dual(cp4d_ctx *ctx, const float *ft_above);
/* Fig. 2 steps 5-6: f <- f - tau K1^T h1 + tau div h2, ft <- f+ + theta (f+ - f).
 * h2z_below: the lower neighbour's LAST slice of the z-component of h2, AFTER that neighbour's cp4d_step_dual of this iteration. */
int cp4d_step_primal(cp4d_ctx *ctx, const float *h2z_below);

/* ---- end-to-end call with HOST buffers (pinned or pageable) ---------------------------------- */
/* H2D copy of g_host (S), reset to zeros, n_iters iterations with the current steps, D2H copy of f
 * into f_host (V).  Syncs. */
int cp4d_solve_host(cp4d_ctx *ctx, const float *g_host, int32_t n_iters, float *f_host);

int cp4d_sync(cp4d_ctx *ctx);
/* number of kernels (and memset nodes) this context has enqueued since create */
int cp4d_launch_count(const cp4d_ctx *ctx, uint64_t *count_out);
/* cp4d_iterate(n >= 2) on a capturable stream (any stream but the legacy default stream 0) captures one iteration of
 * Fig. 2 into a CUDA graph on first use and replays it n times (with the one-pass step: TWO iterations, after which the
 * double-buffered arrays are back in their roles, replayed n / 2 times; an odd iteration is launched directly); the graph is rebuilt when cp4d_set_steps changes tau or
 * sigma, and it is bypassed while cp4d_profile_begin is active (the per-kernel events sit between the launches) and on
 * stream 0, where the launches are issued one by one.  count_out: graph replays since create (each one is counted in
 * cp4d_launch_count with the number of kernels and memset nodes of one iteration). */
int cp4d_graph_replays(const cp4d_ctx *ctx, uint64_t *count_out);
/* "" while cp4d_iterate replays the graph (or has not tried yet); otherwise the reason it launches one by one (legacy
 * stream, or the CUDA error text of the failed capture / instantiation).  The eager path computes the same iterates, so a
 * failed capture is not an error of cp4d_iterate -- but it is never silent. */
const char *cp4d_graph_note(const cp4d_ctx *ctx);

/* ---- per-kernel device timing (CUDA events on the context's stream) ------------- */
/* Kernel classes of the hot path.  FORWARD includes the zero-fill of its partial-sum scratch. */
#define CP4D_K_FORWARD     0  /* ray sums over the base angles, all m coefficients per ray (Eq. 9)       */
#define CP4D_K_SYNTH       1  /* synthesis with Phi + unfold (+ F1* prox, step 3)                         */
#define CP4D_K_FOLD        2  /* analysis with Phi + pi-fold of the sinogram (L204-L212)                  */
#define CP4D_K_BACKPROJECT 3  /* backprojection over the base angles (Eq. 10)                             */
#define CP4D_K_GRAD        4
#define CP4D_K_DIV         5
#define CP4D_K_PROX_F2     6  /* fused grad + projection (step 4)                                         */
#define CP4D_K_UPDATE      7  /* fused div + primal update + over-relaxation (steps 5-6)                  */
#define CP4D_K_REDUCE      8
#define CP4D_K_MISC        9
#define CP4D_K_MIX        10  /* frame mode: per-voxel frame <-> coefficient contraction (L231-L237)           */
#define CP4D_K_PROX_UPDATE 11 /* steps 4-6 in one pass (cp4d_workspace_bytes_fused)                              */
#define CP4D_K_COUNT      12
typedef struct {
    double   ms[CP4D_K_COUNT];        /* summed device time of the class since cp4d_profile_begin       */
    uint64_t launches[CP4D_K_COUNT];  /* timed launches of the class                                      */
} cp4d_profile;
/* Start recording a CUDA event pair around every kernel this context enqueues (clears old records). */
int cp4d_profile_begin(cp4d_ctx *ctx);
/* Sync, stop recording, sum the event pairs per class into *out_host (HOST). */
int cp4d_profile_end(cp4d_ctx *ctx, cp4d_profile *out_host);
const char *cp4d_kernel_name(int kernel_class);
const char *cp4d_strerror(int code);
const char *cp4d_last_error(const cp4d_ctx *ctx);
const char *cp4d_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CP4D_H */
