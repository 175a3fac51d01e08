// Internal declarations of libcp4d.so (sm_100a).  Not part of the C ABI (include/cp4d.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "cp4d.h"

namespace cp4d {

constexpr int TILE = 32;          // voxel tile side of both projector kernels
constexpr int WIN = 48;           // bins a TILE x TILE tile can touch at one angle: floor(31*sqrt2)+4
constexpr int MAX_M = 32;

// per (tile, base angle) geometry, computed in fp64 on the host at create:
// bin coordinate of tile-local voxel (lx, ly) relative to the window start is  delta + lx*c + ly*s.
struct TileGeo {
    int32_t bstart;  // first bin of the tile's window at this angle (may be < 0 or > nd-WIN)
    float delta;     // p(tile origin) - bstart, in [1, WIN)
};

// per base angle, fp32 roundings of the fp64 host values
struct AngleTab {
    float c, s, inv_a;  // cos, sin, 1/max(|c|,|s|)
    int32_t col_step;   // 1: |s| >= |c| (ray steps over columns ix), 0: steps over rows iy
    // forward projector, dominant-axis stepping: the ray with window coordinate du crosses step k at (du - k cc)/ss,
    // (cc, ss) = (c, s) when col_step else (s, c)
    float fw_inv, fw_step, fw_istep;  // 1/ss, -cc/ss, 1/fw_step (0 when |fw_step| < 1e-6), rounded from fp64
};

// forward projector parameters of one base angle, one 16-byte load (see AngleTab::fw_*)
struct FwAngle {
    float inv, step, istep, inv_a;
};

struct FwTable;   // projectors.cu: the forward kernel's per-angle parameters as a kernel parameter (constant bank)

struct Dims {
    int n, nz, nd, na, npi, n0, m, Q;  // Q = m/4 float4 chunks per voxel of a coefficient stack
    int nf, mp, Qp;                    // frame mode: nf frames (0 = coefficient mode); mp = nf ? nf : m is the
                                       // length of the primal 4th axis, Qp = mp/4
    int64_t Vc;                        // elements of a coefficient stack nz*n*n*m (== V in coefficient mode)
    int mb;                            // rows of the caller's basis table phi_host (the paper's M); m above is what the
                                       // projector pair carries per voxel: M, or N_t in collapsed frame mode
    int tiles_1d, tiles;               // ceil(n/TILE), tiles_1d^2
    int64_t V, S;                      // elements of a primal array nz*n*n*mp / a sinogram
    int64_t slice4;                    // float4 per primal slice: n*n*Qp
    int gp, gpl;                       // row pitch / left pad (float4) of the projector scratch: a row holds bins -gpl .. gp-gpl-1
    int64_t scratch4;                  // float4 of projector scratch: nz*n0*Q*gp
};

}  // namespace cp4d

struct cp4d_ctx {
    cp4d::Dims d;
    float lambda1, lambda2, theta;
    int z_open;                  // cp4d_params.z_open: bit 0 lower face interior, bit 1 upper face interior (z-slab of a taller volume)
    float tau, sigma;
    bool have_steps, have_data;
    int device;
    cudaStream_t stream;
    // workspace carve-up (device pointers)
    float *f, *ft, *bp, *h2, *h1, *g, *tmp_s;
    // one-pass step (fused_step.cu): the second copies of ft and h2; cp4d_iterate swaps (ft, ft_alt) and (h2, h2_alt) after every
    // iteration, flip = iterations since the copies were in the roles they had at create, mod 2
    bool fused;
    float *ft_alt, *h2_alt;
    int flip;
    float *cf, *cb, *psi;      // frame mode: coefficient stacks (analysis output, backprojection output), Psi[j][q] = phi_j(t_q)
    float4 *scratch;           // folded sinogram gt of the adjoint: [z][i][jc][gpl + b] float4, pitch gp; the pads stay ZERO (nothing
                               // else may write here), so every tile window of the backprojector is readable and reads 0 off the detector
    float4 *psum;              // forward partial ray sums P[z][i][b][j] (without the 1/a of the base angle, which k_synth applies),
                               // j fastest, no padding: zeroed before, RED'ed by the projector
    float *phi;                // [j][k]
    cp4d::AngleTab *ang;       // [n0]
    cp4d::FwAngle *fwang;      // [n0]
    int32_t *fworder;          // [n0]: base angles whose rays step over columns first, then the others
    int n_colstep;             // how many of the former
    // one CP iteration captured as a CUDA graph (cp4d_iterate replays it; rebuilt when tau / sigma change).  Not available on
    // the legacy default stream, which cannot be captured: the launches are then issued one by one, and `note` says why.
    cudaGraphExec_t iter_graph;
    uint64_t iter_graph_launches, graph_replays;
    bool iter_graph_off;
    cp4d::FwTable *fwtab_host; // host copy of fwang / fworder for the kernel-parameter path (n0 <= 512), else null
    int4 *fw_groups;           // tensor-core forward projector (forward_mma.cu): base angles of each pass in groups of up to four neighbours
    int n_groups0, n_groups1;
    unsigned *fw_items;        // its work items per (tile, pass), built once by cp4d_create (forward_mma_build); null if the shape is not supported
    int2 *fw_counts;           // [tile][pass]: (long, short) items
    int *bm_order;             // its tile order (backproject_mma_order), tiles ints
    void *bm_rec;              // tensor-core backprojector (backproject_mma.cu): angle records per (tile, angle), built once by cp4d_create; null if unsupported
    int fw_mode;               // CP4D_PROJ_AUTO / _FP32 (cp4d_set_projector_mode): both projectors
    int n_cpos;                // the first n_cpos base angles have cos >= 0 (backprojector: chunks never mix the signs)
    cp4d::TileGeo *geo;        // [tile][n0]
    double *red;               // 8 doubles for reductions
    uint64_t launches;
    std::string err;             // text of the last error (cp4d_last_error)
    std::string note;            // why cp4d_iterate is not replaying a CUDA graph, if it is not (cp4d_graph_note)
    // per-kernel event timing (cp4d_profile_begin/end)
    bool prof_on;
    struct ProfRec { int cls; cudaEvent_t a, b; };
    std::vector<ProfRec> prof;       // records of the current profiling window
    std::vector<cudaEvent_t> ev_pool;  // reusable events
};

namespace cp4d {

// RAII event pair around the launches of one kernel class; no-op unless profiling is on
struct ProfScope {
    cp4d_ctx *c;
    cudaEvent_t a, b;
    int cls;
    ProfScope(cp4d_ctx *ctx, int kernel_class) : c(ctx), a(nullptr), b(nullptr), cls(kernel_class) {
        if (!c->prof_on) return;
        a = take(); b = take();
        if (a && b) cudaEventRecord(a, c->stream);
    }
    ~ProfScope() {
        if (!a || !b) return;
        cudaEventRecord(b, c->stream);
        c->prof.push_back({cls, a, b});
    }
    cudaEvent_t take() {
        if (!c->ev_pool.empty()) { cudaEvent_t e = c->ev_pool.back(); c->ev_pool.pop_back(); return e; }
        cudaEvent_t e = nullptr;
        if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        return e;
    }
};

// launchers (each enqueues on ctx->stream and bumps ctx->launches); return cudaError_t
// halo: the neighbour slab's slice (grad / prox: f at z = nz; div / update: p_z at z = -1), null on a closed face
cudaError_t launch_grad(cp4d_ctx *c, const float *f, float *p, const float *halo = nullptr);
cudaError_t launch_div(cp4d_ctx *c, const float *p, float *f, const float *halo = nullptr);
cudaError_t launch_prox_f2(cp4d_ctx *c, float sigma, const float *ft, float *h2, const float *halo = nullptr);
cudaError_t launch_update(cp4d_ctx *c, float tau, const float *bp, const float *h2, float *f, float *ft, const float *halo = nullptr);
cudaError_t launch_fold(cp4d_ctx *c, const float *g, float4 *gt);
// synth: out = K1 f from partial sums P.  mode 0: g_out = v ; mode 1: h1 = (h1 + sigma (v - g))/(1+sigma)
cudaError_t launch_synth(cp4d_ctx *c, const float4 *P, int mode, float sigma, const float *g, float *out);
// host helpers of projectors.cu for cp4d_create / cp4d_destroy
FwTable *fwtable_new(const FwAngle *ang, const int32_t *order, int n0);   // null when n0 is too large
void fwtable_free(FwTable *t);
cudaError_t launch_forward_partial(cp4d_ctx *c, const float *f, float4 *P);
cudaError_t forward_init();        // once per process and device: opt in to the forward kernels' dynamic shared memory
// forward_mma.cu: the tensor-core forward projector (split-bf16 HMMA, fp32 accumulate)
bool forward_mma_supported(const Dims &d);
bool forward_mma_preferred(const Dims &d);     // what CP4D_PROJ_AUTO picks
cudaError_t forward_mma_init();
int forward_mma_groups(const FwAngle *fw, const int32_t *order, int n0, int n_colstep, int4 *out, int *ngroups0, int *ngroups1);
cudaError_t launch_forward_mma(cp4d_ctx *c, const float *f, float *P);
uint64_t forward_mma_item_bytes(const Dims &d);   // workspace bytes of the item slots (0 if the shape is not supported)
bool forward_mma_usable(const cp4d_ctx *c);       // supported shape and the groups fit the kernel's tables
cudaError_t forward_mma_build(cp4d_ctx *c);       // cp4d_create: builds the work items
uint64_t backproject_mma_rec_bytes(const Dims &d);  // workspace bytes of the tensor backprojector's angle records (0 if unsupported)
cudaError_t backproject_mma_build(cp4d_ctx *c);     // cp4d_create: builds them
void backproject_mma_order(int tiles_1d, int *order);  // host: tile order of a launch, tiles_1d^2 entries
// backproject_mma.cu: the tensor-core adjoint (fold into split-bf16 rows + backprojection); same shapes as forward_mma
int backproject_mma_nb16(const Dims &d);
int64_t backproject_mma_scratch_units(const Dims &d);
cudaError_t backproject_mma_init();
cudaError_t backproject22_init();
cudaError_t fused_step_init();
// steps 4-6 of Fig. 2 in one pass: reads ft, h2, bp, f; writes h2_new, ft_new (second copies) and f in place
cudaError_t launch_prox_update(cp4d_ctx *c, float sigma, float tau, const float *ft, const float *h2, float *h2_new,
                               const float *bp, float *f, float *ft_new);
cudaError_t launch_fold_split(cp4d_ctx *c, const float *g, float4 *gt);
cudaError_t launch_backproject_mma(cp4d_ctx *c, const float4 *gt, float *f_out);
cudaError_t launch_backproject(cp4d_ctx *c, const float4 *gt, float *f_out, int Q_override = 0);
// cp4d_fbp: Shepp-Logan filter along the bins; per-half-rotation rows gathered into the projector scratch (box basis)
cudaError_t launch_filter_sl(cp4d_ctx *c, const float *g, float *gf);
cudaError_t launch_fold_halfrot(cp4d_ctx *c, const float *gf, float4 *gt, int Qf, float scale);
// out[v][a] = sum_b T(a,b) in[v][b] per voxel v, T(a,b) = psi[a*sa + b*sb]  (frame <-> coefficient contraction, L231-L237)
cudaError_t launch_mix(cp4d_ctx *c, const float *in, float *out, int na_out, int nb_in, int sa, int sb);
cudaError_t launch_tv_sum(cp4d_ctx *c, const float *f, double *slot);                       // sum |K2 f|_2
cudaError_t launch_kkt_sum(cp4d_ctx *c, const float *bp, const float *h2, double *slot);    // sum (bp - div h2)^2
cudaError_t launch_sumsq_dot(cp4d_ctx *c, const float *x, const float *y, uint64_t n, double *slot);
cudaError_t launch_fill_normal(cp4d_ctx *c, float *x, uint64_t n, uint64_t seed);
// x = (a - b) * scale   (b nullable)
cudaError_t launch_scale_diff(cp4d_ctx *c, float *x, const float *a, const float *b, float scale, uint64_t n);

}  // namespace cp4d
