// C ABI of libcp4d.so (include/cp4d.h): validation, workspace carving, host-side fp64 tables, and the
// stream-ordered orchestration of Fig. 2.  No kernel code here.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "cp4d_internal.cuh"

using namespace cp4d;

namespace {

constexpr uint64_t ALIGN = 256;
inline uint64_t up(uint64_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

int validate(const cp4d_params *p, Dims *d) {
    if (!p) return CP4D_EINVAL;
    if (p->nx != p->ny || p->nx < 2 || p->nz < 1 || p->nd < 2 || p->n_angles < 1 || p->n_half_rot < 1) return CP4D_EINVAL;
    if (p->n_angles % p->n_half_rot) return CP4D_EINVAL;
    if (p->m < 4 || p->m > MAX_M || p->m % 4) return CP4D_EINVAL;
    if (!(p->lambda1 >= 0.f) || !(p->theta_relax >= 0.f && p->theta_relax <= 1.f) || !std::isfinite(p->lambda2)) return CP4D_EINVAL;
    d->n = p->nx; d->nz = p->nz; d->nd = p->nd; d->na = p->n_angles; d->npi = p->n_half_rot;
    d->n0 = d->na / d->npi; d->m = p->m; d->Q = p->m / 4;
    // frame mode (L214-L237): n_frames frames every n_angles/n_frames angles; the primal 4th axis is the frame index
    if (p->n_frames < 0 || (p->n_frames > 0 && (p->n_frames % 4 || p->n_frames > MAX_M || p->n_angles % p->n_frames))) return CP4D_EINVAL;
    if (p->z_open < 0 || p->z_open > 3) return CP4D_EINVAL;
    // k_fold / k_synth keep the n_half_rot x m slice of Phi of their base angle in (default-limit) dynamic shared memory
    if ((int64_t)p->n_half_rot * p->m * 4 > 48 * 1024) return CP4D_EINVAL;
    d->nf = p->n_frames; d->mp = d->nf ? d->nf : d->m; d->Qp = d->mp / 4;
    d->mb = p->m;
    // Collapsed frame mode (N_t <= M): K1 o A = sum_q W[k,q] R f(t_q) with W[k,q] = sum_j phi_j(t_k) phi_j(t_q), so the projector
    // pair can carry the N_t frames themselves with the N_t x N_theta table W^T in place of Phi: no analysis pass, N_t/M of the
    // projector work.  From here on it is a coefficient-mode problem with m = N_t (cp4d_create builds the table).
    if (d->nf && d->nf <= d->m) { d->m = d->nf; d->Q = d->nf / 4; d->nf = 0; }
    d->tiles_1d = (d->n + TILE - 1) / TILE; d->tiles = d->tiles_1d * d->tiles_1d;
    d->V = (int64_t)d->nz * d->n * d->n * d->mp;
    d->Vc = (int64_t)d->nz * d->n * d->n * d->m;
    d->S = (int64_t)d->nz * d->na * d->nd;
    d->slice4 = (int64_t)d->n * d->n * d->Qp;
    // pads of the scratch rows: the window [bstart, bstart + WIN + 8) of a 32x32 tile (edge tiles reach past the grid) may
    // leave the detector by at most sqrt2 * E - (nd-1)/2 + 2 bins, E = largest |coordinate| a tile covers
    // (cp4d_create checks the exact values)
    const double cen0 = 0.5 * (d->n - 1), ext = std::fmax(cen0, (double)d->tiles_1d * TILE - 1.0 - cen0);
    const int over = (int)std::ceil(std::fmax(0.0, 1.41421356237309515 * ext - 0.5 * (d->nd - 1))) + 3;
    d->gpl = over;
    d->gp = d->nd + 2 * over + WIN + 8;
    if (d->gp % 8 == 0) d->gp += 1;   // a pitch of whole 128-byte lines measured 1 % slower in the forward projector's REDs
    d->scratch4 = (int64_t)d->nz * d->n0 * d->Q * d->gp;
    if (forward_mma_supported(*d)) d->scratch4 = std::max(d->scratch4, backproject_mma_scratch_units(*d));   // split-bf16 rows, whole z-groups
    if (d->nz > 65535 || d->tiles > 2000000) return CP4D_EINVAL;
    return CP4D_OK;
}

struct Carve {
    uint64_t ft_alt, h2_alt;
    uint64_t f, ft, bp, h2, h1, g, tmp_s, scratch, psum, phi, ang, geo, red, cf, cb, psi, fwang, fworder, fwpairs, fwitems, fwcounts, bmrec, bmorder, total;
};
Carve carve(const Dims &d, bool fused = false) {
    Carve c;
    uint64_t o = 0;
    auto take = [&](uint64_t bytes) { uint64_t r = o; o += up(bytes); return r; };
    c.f = take(d.V * 4); c.ft = take(d.V * 4); c.bp = take(d.V * 4); c.h2 = take(d.V * 16);
    c.h1 = take(d.S * 4); c.g = take(d.S * 4); c.tmp_s = take(d.S * 4); c.scratch = take(d.scratch4 * 16);
    c.psum = take((uint64_t)d.nz * d.n0 * d.nd * d.m * 4);
    c.phi = take((uint64_t)d.m * d.na * 4); c.ang = take((uint64_t)d.n0 * sizeof(AngleTab));
    c.geo = take((uint64_t)d.tiles * d.n0 * sizeof(TileGeo)); c.red = take(64);
    c.fwang = take((uint64_t)d.n0 * sizeof(FwAngle)); c.fworder = take((uint64_t)d.n0 * 4);
    c.fwpairs = take((uint64_t)d.n0 * sizeof(int4));
    c.fwitems = take(forward_mma_item_bytes(d)); c.fwcounts = take((uint64_t)d.tiles * 2 * sizeof(int2));
    c.bmrec = take(backproject_mma_rec_bytes(d)); c.bmorder = take((uint64_t)d.tiles * sizeof(int));
    c.cf = c.cb = c.psi = 0;
    if (d.nf) { c.cf = take(d.Vc * 4); c.cb = take(d.Vc * 4); c.psi = take((uint64_t)d.mb * d.nf * 4); }
    c.ft_alt = c.h2_alt = 0;
    if (fused) { c.ft_alt = take(d.V * 4); c.h2_alt = take(d.V * 16); }
    c.total = o;
    return c;
}

int fail(cp4d_ctx *c, int code, const char *what, cudaError_t e = cudaSuccess) {
    if (c) {
        c->err = what;
        if (e != cudaSuccess) { c->err += ": "; c->err += cudaGetErrorString(e); }
    }
    return code;
}
#define CK(call, what)                                                  \
    do {                                                                \
        cudaError_t e__ = (call);                                       \
        if (e__ != cudaSuccess) return fail(ctx, CP4D_ECUDA, what, e__); \
    } while (0)

// Every entry point runs with the context's device current and puts the caller's device back on exit: a context made for
// device 1 works whatever device the calling thread has selected (streams, events and launches are per device).
struct DevGuard {
    int prev = -1;
    explicit DevGuard(int dev) {
        int cur = -1;
        if (cudaGetDevice(&cur) != cudaSuccess) { cudaGetLastError(); cur = -1; }
        if (cur != dev && cudaSetDevice(dev) == cudaSuccess) prev = cur;
    }
    ~DevGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
    DevGuard(const DevGuard &) = delete;
    DevGuard &operator=(const DevGuard &) = delete;
};

bool overlap(const void *a, uint64_t na, const void *b, uint64_t nb) {
    const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
    return x < y + nb && y < x + na;
}
bool bad_ptr(const void *p) { return !p || ((uintptr_t)p & 15); }

// f is primal-shaped: the coefficient stack, or (frame mode) the frames, analysed into ctx->cf first
int forward_into(cp4d_ctx *ctx, const float *f, int mode, float sigma, const float *g, float *out) {
    if (ctx->d.nf) {
        CK(launch_mix(ctx, f, ctx->cf, ctx->d.m, ctx->d.nf, ctx->d.nf, 1), "analysis");     // (here m == mb)    // T(j,q) = psi[j*nf + q]
        f = ctx->cf;
    }
    CK(launch_forward_partial(ctx, f, ctx->psum), "forward_partial");
    CK(launch_synth(ctx, ctx->psum, mode, sigma, g, out), "synth");
    return CP4D_OK;
}
int adjoint_into(cp4d_ctx *ctx, const float *g, float *f) {
    // the tensor-core pair where it is asked for, and in auto mode where the problem fills the GPU (there it is the faster one)
    if (forward_mma_usable(ctx) && (ctx->fw_mode == CP4D_PROJ_TENSOR || (ctx->fw_mode == CP4D_PROJ_AUTO && forward_mma_preferred(ctx->d)))) {
        CK(launch_fold_split(ctx, g, ctx->scratch), "fold");
        CK(launch_backproject_mma(ctx, ctx->scratch, ctx->d.nf ? ctx->cb : f), "backproject");
    } else {
        CK(launch_fold(ctx, g, ctx->scratch), "fold");
        CK(launch_backproject(ctx, ctx->scratch, ctx->d.nf ? ctx->cb : f), "backproject");
    }
    if (ctx->d.nf) CK(launch_mix(ctx, ctx->cb, f, ctx->d.nf, ctx->d.m, 1, ctx->d.nf), "analysis^T");  // T(q,j) = psi[j*nf + q]
    return CP4D_OK;
}

}  // namespace

extern "C" {

const char *cp4d_version(void) { return "cp4d 0.1 (sm_100a)"; }

const char *cp4d_strerror(int code) {
    switch (code) {
    case CP4D_OK: return "ok";
    case CP4D_EINVAL: return "invalid argument";
    case CP4D_EWORKSPACE: return "workspace missing or too small";
    case CP4D_EUNSUPPORTED: return "no sm_100 CUDA device";
    case CP4D_ECUDA: return "CUDA error";
    case CP4D_ESTATE: return "call order: set_data/set_steps before iterate";
    case CP4D_ENOMEM: return "host allocation failed";
    case CP4D_EINTERNAL: return "internal invariant violated (scratch window)";
    case CP4D_ETOOLARGE: return "problem exceeds the static scratch array (CP4D_STATIC_SCRATCH_BYTES)";
    default: return "unknown error";
    }
}

const char *cp4d_last_error(const cp4d_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int cp4d_workspace_bytes(const cp4d_params *p, uint64_t *out) {
    Dims d;
    if (!out) return CP4D_EINVAL;
    int r = validate(p, &d);
    if (r) return r;
    *out = carve(d).total;
    return CP4D_OK;
}

int cp4d_workspace_bytes_fused(const cp4d_params *p, uint64_t *out) {
    Dims d;
    if (!out) return CP4D_EINVAL;
    int r = validate(p, &d);
    if (r) return r;
    *out = carve(d, true).total;
    return CP4D_OK;
}

int cp4d_fused_step_in_use(const cp4d_ctx *ctx, int32_t *out) {
    if (!ctx || !out) return CP4D_EINVAL;
    *out = ctx->fused ? 1 : 0;
    return CP4D_OK;
}

int cp4d_create(const cp4d_params *p, cp4d_ctx **out) {
    if (!out) return CP4D_EINVAL;
    *out = nullptr;
    Dims d;
    int r = validate(p, &d);
    if (r) return r;
    if (!p->phi_host) return CP4D_EINVAL;
    // a whole-volume context on a workspace with room for the second copies of ft and h2 runs steps 4-6 as one pass
    const bool fused = p->z_open == 0 && d.slice4 < (int64_t)1 << 31 && p->workspace_dev && p->workspace_bytes >= carve(d, true).total;
    const Carve cv = carve(d, fused);
    if (!p->workspace_dev || p->workspace_bytes < cv.total) return CP4D_EWORKSPACE;
    if ((uintptr_t)p->workspace_dev & (ALIGN - 1)) return CP4D_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || p->device < 0 || p->device >= ndev) { cudaGetLastError(); return CP4D_EUNSUPPORTED; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, p->device) != cudaSuccess || prop.major != 10) { cudaGetLastError(); return CP4D_EUNSUPPORTED; }
    DevGuard dev_guard(p->device);     // the caller's current device is restored on return
    {
        int cur = -1;
        if (cudaGetDevice(&cur) != cudaSuccess || cur != p->device) { cudaGetLastError(); return CP4D_ECUDA; }
    }
    if (forward_init() != cudaSuccess || backproject_mma_init() != cudaSuccess || backproject22_init() != cudaSuccess || fused_step_init() != cudaSuccess) { cudaGetLastError(); return CP4D_ECUDA; }

    cp4d_ctx *ctx = new (std::nothrow) cp4d_ctx();
    if (!ctx) return CP4D_ENOMEM;
    ctx->d = d; ctx->lambda1 = p->lambda1; ctx->lambda2 = p->lambda2; ctx->theta = p->theta_relax; ctx->z_open = p->z_open;
    ctx->tau = ctx->sigma = 0.f; ctx->have_steps = ctx->have_data = false;
    ctx->device = p->device; ctx->stream = (cudaStream_t)p->stream; ctx->launches = 0; ctx->prof_on = false;
    ctx->fwtab_host = nullptr;
    ctx->iter_graph = nullptr; ctx->iter_graph_launches = 0; ctx->graph_replays = 0; ctx->iter_graph_off = false;
    char *w = (char *)p->workspace_dev;
    ctx->f = (float *)(w + cv.f); ctx->ft = (float *)(w + cv.ft); ctx->bp = (float *)(w + cv.bp);
    ctx->h2 = (float *)(w + cv.h2); ctx->h1 = (float *)(w + cv.h1); ctx->g = (float *)(w + cv.g);
    ctx->tmp_s = (float *)(w + cv.tmp_s);
    ctx->fused = fused; ctx->flip = 0;
    ctx->ft_alt = fused ? (float *)(w + cv.ft_alt) : nullptr; ctx->h2_alt = fused ? (float *)(w + cv.h2_alt) : nullptr;
    ctx->fwang = (FwAngle *)(w + cv.fwang); ctx->fworder = (int32_t *)(w + cv.fworder);
    ctx->fw_groups = (int4 *)(w + cv.fwpairs); ctx->fw_mode = CP4D_PROJ_AUTO;
    ctx->fw_items = forward_mma_item_bytes(d) ? (unsigned *)(w + cv.fwitems) : nullptr; ctx->fw_counts = (int2 *)(w + cv.fwcounts);
    ctx->bm_rec = backproject_mma_rec_bytes(d) ? (void *)(w + cv.bmrec) : nullptr; ctx->bm_order = (int *)(w + cv.bmorder);
    ctx->cf = d.nf ? (float *)(w + cv.cf) : nullptr; ctx->cb = d.nf ? (float *)(w + cv.cb) : nullptr;
    ctx->psi = d.nf ? (float *)(w + cv.psi) : nullptr;
    ctx->scratch = (float4 *)(w + cv.scratch); ctx->psum = (float4 *)(w + cv.psum); ctx->phi = (float *)(w + cv.phi);
    ctx->ang = (AngleTab *)(w + cv.ang); ctx->geo = (TileGeo *)(w + cv.geo); ctx->red = (double *)(w + cv.red);

    // host prologue: fp64 angle tables and per-(tile, angle) window geometry
    std::vector<AngleTab> ang(d.n0);
    std::vector<double> cs(2 * (size_t)d.n0);
    const double PI = 3.14159265358979323846264338327950288;
    for (int i = 0; i < d.n0; ++i) {
        const double th = (double)i * PI / (double)d.n0, c = std::cos(th), s = std::sin(th);
        cs[2 * i] = c; cs[2 * i + 1] = s;
        ang[i].c = (float)c; ang[i].s = (float)s;
        ang[i].inv_a = (float)(1.0 / std::fmax(std::fabs(c), std::fabs(s)));
        ang[i].col_step = std::fabs(s) >= std::fabs(c) ? 1 : 0;
        {
            const double cc = ang[i].col_step ? c : s, ss = ang[i].col_step ? s : c, st = -cc / ss;
            ang[i].fw_inv = (float)(1.0 / ss); ang[i].fw_step = (float)st;
            ang[i].fw_istep = std::fabs(st) < 1e-6 ? 0.0f : (float)(1.0 / st);
        }
    }
    ctx->n_cpos = 0;
    while (ctx->n_cpos < d.n0 && ang[ctx->n_cpos].c >= 0.f) ++ctx->n_cpos;
    for (int i = ctx->n_cpos; i < d.n0; ++i)
        if (ang[i].c >= 0.f) { delete ctx; return CP4D_EINTERNAL; }   // cos is monotone on [0, pi): cannot happen
    std::vector<FwAngle> fwang(d.n0);
    std::vector<int32_t> fworder;
    for (int pass = 0; pass < 2; ++pass) {
        for (int i = 0; i < d.n0; ++i)
            if ((ang[i].col_step != 0) == (pass == 0)) fworder.push_back(i);
        if (pass == 0) ctx->n_colstep = (int)fworder.size();
    }
    for (int i = 0; i < d.n0; ++i) fwang[i] = FwAngle{ang[i].fw_inv, ang[i].fw_step, ang[i].fw_istep, ang[i].inv_a};
    ctx->fwtab_host = fwtable_new(fwang.data(), fworder.data(), d.n0);
    std::vector<int4> fwpairs(d.n0);
    forward_mma_groups(fwang.data(), fworder.data(), d.n0, ctx->n_colstep, fwpairs.data(), &ctx->n_groups0, &ctx->n_groups1);
    std::vector<TileGeo> geo((size_t)d.tiles * d.n0);
    const double cen = 0.5 * (d.n - 1), cd = 0.5 * (d.nd - 1);
    for (int t = 0; t < d.tiles; ++t) {
        const double x0 = (double)(t % d.tiles_1d) * TILE - cen, y0 = (double)(t / d.tiles_1d) * TILE - cen;
        for (int i = 0; i < d.n0; ++i) {
            // the tables hold the fp32-rounded c, s the kernels multiply lx, ly with; the tile origin term is fp64
            const double c = cs[2 * i], s = cs[2 * i + 1];
            const double p0 = x0 * c + y0 * s + cd;
            const double pmin = p0 + std::fmin(0.0, (TILE - 1) * c) + std::fmin(0.0, (TILE - 1) * s);
            const double bs = std::floor(pmin) - 1.0;
            geo[(size_t)t * d.n0 + i].bstart = (int32_t)bs;
            // validate() sized the pads of the scratch rows for this: cannot happen
            if ((int32_t)bs < -d.gpl || (int32_t)bs + WIN + 8 > d.gp - d.gpl) { cp4d_destroy(ctx); return CP4D_EINTERNAL; }
            geo[(size_t)t * d.n0 + i].delta = (float)(p0 - bs);
        }
    }
    // frame mode: Psi[j][q] = phi_j(t_q), t_q the time of angle q * n_angles / n_frames (L231-L237: f_j = sum_q f(t_q) phi_j(t_q))
    const int ntf = p->n_frames, fstride = ntf ? d.na / ntf : 0;
    std::vector<float> psi((size_t)d.mb * (d.nf ? d.nf : 1));
    for (int j = 0; j < d.mb && d.nf; ++j)
        for (int q = 0; q < d.nf; ++q) psi[(size_t)j * d.nf + q] = p->phi_host[(size_t)j * d.na + (size_t)q * fstride];
    // the table the projector pair uses: Phi itself, or in collapsed frame mode W^T[q][k] = sum_j phi_j(t_q) phi_j(t_k) (fp64 sums)
    std::vector<float> phi_eff((size_t)d.m * d.na);
    const bool collapsed = ntf > 0 && d.nf == 0;
    for (int r = 0; r < d.m; ++r)
        for (int k = 0; k < d.na; ++k) {
            if (!collapsed) { phi_eff[(size_t)r * d.na + k] = p->phi_host[(size_t)r * d.na + k]; continue; }
            double acc = 0.0;
            for (int j = 0; j < d.mb; ++j) acc += (double)p->phi_host[(size_t)j * d.na + (size_t)r * fstride] * (double)p->phi_host[(size_t)j * d.na + k];
            phi_eff[(size_t)r * d.na + k] = (float)acc;
        }
    std::vector<int> bmorder(d.tiles);
    backproject_mma_order((d.n + TILE - 1) / TILE, bmorder.data());
    cudaError_t e;
    if ((d.nf && (e = cudaMemcpyAsync(ctx->psi, psi.data(), psi.size() * 4, cudaMemcpyHostToDevice, ctx->stream)) != cudaSuccess) ||
        (e = cudaMemcpyAsync(ctx->phi, phi_eff.data(), (size_t)d.m * d.na * 4, cudaMemcpyHostToDevice, ctx->stream)) != cudaSuccess ||
        (e = cudaMemcpyAsync(ctx->ang, ang.data(), ang.size() * sizeof(AngleTab), cudaMemcpyHostToDevice, ctx->stream)) != cudaSuccess ||
        (e = cudaMemcpyAsync(ctx->fwang, fwang.data(), fwang.size() * sizeof(FwAngle), cudaMemcpyHostToDevice, ctx->stream)) != cudaSuccess ||
        (e = cudaMemcpyAsync(ctx->fworder, fworder.data(), fworder.size() * 4, cudaMemcpyHostToDevice, ctx->stream)) != cudaSuccess ||
        (e = cudaMemcpyAsync(ctx->fw_groups, fwpairs.data(), fwpairs.size() * sizeof(int4), cudaMemcpyHostToDevice, ctx->stream)) != cudaSuccess ||
        (e = cudaMemcpyAsync(ctx->bm_order, bmorder.data(), bmorder.size() * sizeof(int), cudaMemcpyHostToDevice, ctx->stream)) != cudaSuccess ||
        (e = cudaMemcpyAsync(ctx->geo, geo.data(), geo.size() * sizeof(TileGeo), cudaMemcpyHostToDevice, ctx->stream)) != cudaSuccess ||
        (e = cudaMemsetAsync(ctx->scratch, 0, (size_t)d.scratch4 * 16, ctx->stream)) != cudaSuccess ||
        (e = forward_mma_build(ctx)) != cudaSuccess ||
        (e = backproject_mma_build(ctx)) != cudaSuccess ||
        (e = cudaStreamSynchronize(ctx->stream)) != cudaSuccess) {
        ctx->err = cudaGetErrorString(e);   // (the context dies with the error: the caller only sees CP4D_ECUDA)
        cudaGetLastError();
        cp4d_destroy(ctx);
        return CP4D_ECUDA;
    }
    *out = ctx;
    return CP4D_OK;
}

int cp4d_destroy(cp4d_ctx *ctx) {
    if (ctx) {
        DevGuard dev_guard(ctx->device);
        for (auto &r : ctx->prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
        for (auto e : ctx->ev_pool) cudaEventDestroy(e);
        fwtable_free(ctx->fwtab_host);
        if (ctx->iter_graph) cudaGraphExecDestroy(ctx->iter_graph);
    }
    delete ctx;
    return CP4D_OK;
}

int cp4d_forward(cp4d_ctx *ctx, const float *f, float *g) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (bad_ptr(f) || bad_ptr(g) || overlap(f, ctx->d.V * 4, g, ctx->d.S * 4)) return fail(ctx, CP4D_EINVAL, "forward: bad pointers");
    return forward_into(ctx, f, 0, 0.f, nullptr, g);
}

int cp4d_adjoint(cp4d_ctx *ctx, const float *g, float *f) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (bad_ptr(f) || bad_ptr(g) || overlap(f, ctx->d.V * 4, g, ctx->d.S * 4)) return fail(ctx, CP4D_EINVAL, "adjoint: bad pointers");
    return adjoint_into(ctx, g, f);
}

int cp4d_grad(cp4d_ctx *ctx, const float *f, float *p) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (ctx->z_open) return fail(ctx, CP4D_ESTATE, "grad: z-slab context, use the *_slab / cp4d_step_* calls");
    if (bad_ptr(f) || bad_ptr(p) || overlap(f, ctx->d.V * 4, p, ctx->d.V * 16)) return fail(ctx, CP4D_EINVAL, "grad: bad pointers");
    CK(launch_grad(ctx, f, p), "grad");
    return CP4D_OK;
}

int cp4d_div(cp4d_ctx *ctx, const float *p, float *f) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (ctx->z_open) return fail(ctx, CP4D_ESTATE, "div: z-slab context, use the *_slab / cp4d_step_* calls");
    if (bad_ptr(f) || bad_ptr(p) || overlap(f, ctx->d.V * 4, p, ctx->d.V * 16)) return fail(ctx, CP4D_EINVAL, "div: bad pointers");
    CK(launch_div(ctx, p, f), "div");
    return CP4D_OK;
}

int cp4d_prox_f1(cp4d_ctx *ctx, float sigma, const float *ft, const float *g, float *h1) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    const uint64_t Vb = ctx->d.V * 4, Sb = ctx->d.S * 4;
    if (bad_ptr(ft) || bad_ptr(g) || bad_ptr(h1) || overlap(ft, Vb, h1, Sb) || overlap(g, Sb, h1, Sb) || !(sigma > 0.f))
        return fail(ctx, CP4D_EINVAL, "prox_f1: bad arguments");
    return forward_into(ctx, ft, 1, sigma, g, h1);
}

int cp4d_prox_f2(cp4d_ctx *ctx, float sigma, const float *ft, float *h2) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (ctx->z_open) return fail(ctx, CP4D_ESTATE, "prox_f2: z-slab context, use the *_slab / cp4d_step_* calls");
    if (bad_ptr(ft) || bad_ptr(h2) || overlap(ft, ctx->d.V * 4, h2, ctx->d.V * 16)) return fail(ctx, CP4D_EINVAL, "prox_f2: bad pointers");
    CK(launch_prox_f2(ctx, sigma, ft, h2), "prox_f2");
    return CP4D_OK;
}

int cp4d_primal_update(cp4d_ctx *ctx, float tau, const float *h1, const float *h2, float *f, float *ft) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (ctx->z_open) return fail(ctx, CP4D_ESTATE, "primal_update: z-slab context, use the *_slab / cp4d_step_* calls");
    const uint64_t Vb = ctx->d.V * 4, Sb = ctx->d.S * 4;
    if (bad_ptr(h1) || bad_ptr(h2) || bad_ptr(f) || bad_ptr(ft) || overlap(f, Vb, ft, Vb) || overlap(f, Vb, h2, 4 * Vb) ||
        overlap(ft, Vb, h2, 4 * Vb) || overlap(h1, Sb, f, Vb) || overlap(h1, Sb, ft, Vb))
        return fail(ctx, CP4D_EINVAL, "primal_update: bad pointers");
    int r = adjoint_into(ctx, h1, ctx->bp);
    if (r) return r;
    CK(launch_update(ctx, tau, ctx->bp, h2, f, ft), "update");
    return CP4D_OK;
}

int cp4d_dot(cp4d_ctx *ctx, const float *x, const float *y, uint64_t n, double *out) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (bad_ptr(x) || bad_ptr(y) || !out) return fail(ctx, CP4D_EINVAL, "dot: bad pointers");
    CK(launch_sumsq_dot(ctx, x, y, n, ctx->red), "dot");
    CK(cudaMemcpyAsync(out, ctx->red, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream), "dot copy");
    CK(cudaStreamSynchronize(ctx->stream), "dot sync");
    return CP4D_OK;
}

// power iteration from the start vector in ctx->ft
static int norm_from_ft(cp4d_ctx *ctx, int32_t n_iters, float *L_out) {
    const Dims &d = ctx->d;
    float *x = ctx->ft, *y1 = ctx->bp, *y2 = ctx->f;
    double v = 0.0, L = 0.0;
    ctx->have_data = false;  // state buffers are used as scratch
    if (int r = cp4d_dot(ctx, x, x, d.V, &v)) return r;
    if (!(v > 0.0) || !std::isfinite(v)) return fail(ctx, CP4D_EINVAL, "norm: the start vector is zero or not finite");
    CK(launch_scale_diff(ctx, x, x, nullptr, (float)(1.0 / std::sqrt(v)), d.V), "scale");
    for (int it = 0; it < n_iters; ++it) {
        if (int r = forward_into(ctx, x, 0, 0.f, nullptr, ctx->h1)) return r;   // K1 x
        if (int r = adjoint_into(ctx, ctx->h1, y1)) return r;                   // K1^T K1 x
        CK(launch_grad(ctx, x, ctx->h2), "grad");
        CK(launch_div(ctx, ctx->h2, y2), "div");                                // -K2^T K2 x
        CK(launch_scale_diff(ctx, y1, y1, y2, 1.0f, d.V), "diff");              // y = K^T K x
        if (int r = cp4d_dot(ctx, y1, y1, d.V, &v)) return r;
        const double ny = std::sqrt(v);
        L = std::sqrt(ny);                                                      // |x| = 1
        if (!(ny > 0.0)) break;
        CK(launch_scale_diff(ctx, x, y1, nullptr, (float)(1.0 / ny), d.V), "normalise");
    }
    *L_out = (float)L;
    return CP4D_OK;
}

int cp4d_norm(cp4d_ctx *ctx, int32_t n_iters, uint64_t seed, float *L_out) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (ctx->z_open) return fail(ctx, CP4D_ESTATE, "norm: z-slab context, use the *_slab / cp4d_step_* calls");
    if (!L_out || n_iters < 1) return fail(ctx, CP4D_EINVAL, "norm: bad arguments");
    CK(launch_fill_normal(ctx, ctx->ft, ctx->d.V, seed), "fill");
    return norm_from_ft(ctx, n_iters, L_out);
}

int cp4d_norm_start(cp4d_ctx *ctx, int32_t n_iters, const float *x0, float *L_out) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (ctx->z_open) return fail(ctx, CP4D_ESTATE, "norm_start: z-slab context, use the *_slab / cp4d_step_* calls");
    if (!L_out || n_iters < 1 || bad_ptr(x0)) return fail(ctx, CP4D_EINVAL, "norm_start: bad arguments");
    CK(cudaMemcpyAsync(ctx->ft, x0, ctx->d.V * 4, cudaMemcpyDeviceToDevice, ctx->stream), "norm_start copy");
    return norm_from_ft(ctx, n_iters, L_out);
}

int cp4d_set_data(cp4d_ctx *ctx, const float *g) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (bad_ptr(g)) return fail(ctx, CP4D_EINVAL, "set_data: bad pointer");
    CK(cudaMemcpyAsync(ctx->g, g, ctx->d.S * 4, cudaMemcpyDeviceToDevice, ctx->stream), "set_data");
    ctx->have_data = true;
    return CP4D_OK;
}

int cp4d_set_steps(cp4d_ctx *ctx, float tau, float sigma) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (!(tau > 0.f) || !(sigma > 0.f)) return fail(ctx, CP4D_EINVAL, "set_steps: tau, sigma must be > 0");
    if (ctx->iter_graph && (tau != ctx->tau || sigma != ctx->sigma)) {   // the step sizes are baked into the captured launches
        cudaGraphExecDestroy(ctx->iter_graph);
        ctx->iter_graph = nullptr;
    }
    ctx->tau = tau; ctx->sigma = sigma; ctx->have_steps = true;
    return CP4D_OK;
}

int cp4d_reset(cp4d_ctx *ctx, const float *f0) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    const Dims &d = ctx->d;
    if (f0) {
        if (bad_ptr(f0)) return fail(ctx, CP4D_EINVAL, "reset: bad pointer");
        CK(cudaMemcpyAsync(ctx->f, f0, d.V * 4, cudaMemcpyDeviceToDevice, ctx->stream), "reset f");
        CK(cudaMemcpyAsync(ctx->ft, f0, d.V * 4, cudaMemcpyDeviceToDevice, ctx->stream), "reset ft");
    } else {
        CK(cudaMemsetAsync(ctx->f, 0, d.V * 4, ctx->stream), "reset f");
        CK(cudaMemsetAsync(ctx->ft, 0, d.V * 4, ctx->stream), "reset ft");
    }
    CK(cudaMemsetAsync(ctx->h1, 0, d.S * 4, ctx->stream), "reset h1");
    CK(cudaMemsetAsync(ctx->h2, 0, d.V * 16, ctx->stream), "reset h2");
    return CP4D_OK;
}

// one pass of Fig. 2, enqueued on the context's stream
static int iterate_once(cp4d_ctx *ctx) {
    // step 3: h1 <- prox_{sigma F1*}(h1 + sigma K1 ft)
    if (int r = forward_into(ctx, ctx->ft, 1, ctx->sigma, ctx->g, ctx->h1)) return r;
    if (ctx->fused) {
        // steps 4-6 in one pass over the volume, into the second copies of h2 and ft, which then take over
        if (int r = adjoint_into(ctx, ctx->h1, ctx->bp)) return r;
        CK(launch_prox_update(ctx, ctx->sigma, ctx->tau, ctx->ft, ctx->h2, ctx->h2_alt, ctx->bp, ctx->f, ctx->ft_alt), "prox_update");
        std::swap(ctx->ft, ctx->ft_alt); std::swap(ctx->h2, ctx->h2_alt); ctx->flip ^= 1;
        return CP4D_OK;
    }
    // step 4: h2 <- prox_{sigma F2*}(h2 + sigma K2 ft)
    CK(launch_prox_f2(ctx, ctx->sigma, ctx->ft, ctx->h2), "prox_f2");
    // steps 5-6: f <- f - tau K1^T h1 + tau div h2 ; ft <- f+ + theta (f+ - f)
    if (int r = adjoint_into(ctx, ctx->h1, ctx->bp)) return r;
    CK(launch_update(ctx, ctx->tau, ctx->bp, ctx->h2, ctx->f, ctx->ft), "update");
    return CP4D_OK;
}

// capture one iteration into ctx->iter_graph; false (and eager launches from then on) if the stream cannot be captured
static bool capture_iteration(cp4d_ctx *ctx) {
    if (ctx->iter_graph_off) return false;
    if (ctx->stream == nullptr || ctx->stream == cudaStreamLegacy) {
        ctx->note = "the legacy default stream cannot be captured: launches are issued one by one";
        ctx->iter_graph_off = true;
        return false;
    }
    const uint64_t l0 = ctx->launches;
    cudaError_t ce = cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal);
    if (ce != cudaSuccess) {
        cudaGetLastError();
        ctx->note = std::string("cudaStreamBeginCapture failed (") + cudaGetErrorString(ce) + "): launches are issued one by one";
        ctx->iter_graph_off = true;
        return false;
    }
    int r = iterate_once(ctx);
    if (ctx->fused && r == CP4D_OK) r = iterate_once(ctx);      // two iterations: the double-buffered arrays are back in their roles
    cudaGraph_t g = nullptr;
    const cudaError_t e = cudaStreamEndCapture(ctx->stream, &g);
    ctx->iter_graph_launches = ctx->launches - l0;
    ctx->launches = l0;
    bool ok = r == CP4D_OK && e == cudaSuccess && g != nullptr;
    cudaError_t ie = cudaSuccess;
    if (ok) ok = (ie = cudaGraphInstantiate(&ctx->iter_graph, g, 0)) == cudaSuccess;
    if (g) cudaGraphDestroy(g);
    if (!ok) {
        cudaGetLastError();
        // not an error of cp4d_iterate (the eager path computes the same iterates), but never silent: cp4d_graph_note tells why
        ctx->note = "graph capture of one iteration failed (" +
                    (r != CP4D_OK ? "a launch failed during capture: " + ctx->err
                                  : std::string(cudaGetErrorString(e != cudaSuccess ? e : ie))) + "): launches are issued one by one";
        ctx->iter_graph = nullptr;
        ctx->iter_graph_off = true;
        ctx->err.clear();
    }
    return ok;
}

int cp4d_iterate(cp4d_ctx *ctx, int32_t n_iters) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (ctx->z_open) return fail(ctx, CP4D_ESTATE, "iterate: z-slab context, use the *_slab / cp4d_step_* calls");
    if (n_iters < 0) return fail(ctx, CP4D_EINVAL, "iterate: n_iters < 0");
    if (!ctx->have_steps || !ctx->have_data) return fail(ctx, CP4D_ESTATE, "iterate: set_data and set_steps first");
    // the per-kernel timing of cp4d_profile_begin records events between the launches, so it takes the eager path
    int it = 0;
    const int per = ctx->fused ? 2 : 1;                      // iterations per replay
    bool graph = !ctx->prof_on && n_iters >= 2;
    if (graph && ctx->fused && ctx->flip) {                  // the graph holds the launches of flip == 0
        if (int r = iterate_once(ctx)) return r;
        ++it;
    }
    graph = graph && n_iters - it >= per && (ctx->iter_graph || capture_iteration(ctx));
    while (it < n_iters) {
        if (graph && n_iters - it >= per) {
            CK(cudaGraphLaunch(ctx->iter_graph, ctx->stream), "iterate (graph)");
            ctx->launches += ctx->iter_graph_launches;
            ctx->graph_replays++;
            it += per;
        } else {
            if (int r = iterate_once(ctx)) return r;
            ++it;
        }
    }
    return CP4D_OK;
}

// ---- z-slab contexts ----
static int check_halos(cp4d_ctx *ctx, const void *above, const void *below, bool need_above, bool need_below, const char *what) {
    if ((need_above && ((ctx->z_open & 2) != 0) != (above != nullptr)) || (need_below && ((ctx->z_open & 1) != 0) != (below != nullptr)) ||
        (above && bad_ptr(above)) || (below && bad_ptr(below)))
        return fail(ctx, CP4D_EINVAL, what);
    return CP4D_OK;
}

int cp4d_set_z_open(cp4d_ctx *ctx, int32_t z_open) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (z_open < 0 || z_open > 3) return fail(ctx, CP4D_EINVAL, "set_z_open: flags are 0..3");
    ctx->z_open = z_open;
    return CP4D_OK;
}

int cp4d_grad_slab(cp4d_ctx *ctx, const float *f, const float *f_above, float *p) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (bad_ptr(f) || bad_ptr(p) || overlap(f, ctx->d.V * 4, p, ctx->d.V * 16)) return fail(ctx, CP4D_EINVAL, "grad_slab: bad pointers");
    if (int r = check_halos(ctx, f_above, nullptr, true, false, "grad_slab: a halo slice is needed exactly on an interior face")) return r;
    CK(launch_grad(ctx, f, p, f_above), "grad");
    return CP4D_OK;
}

int cp4d_div_slab(cp4d_ctx *ctx, const float *p, const float *pz_below, float *f) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (bad_ptr(f) || bad_ptr(p) || overlap(f, ctx->d.V * 4, p, ctx->d.V * 16)) return fail(ctx, CP4D_EINVAL, "div_slab: bad pointers");
    if (int r = check_halos(ctx, nullptr, pz_below, false, true, "div_slab: a halo slice is needed exactly on an interior face")) return r;
    CK(launch_div(ctx, p, f, pz_below), "div");
    return CP4D_OK;
}

int cp4d_step_dual(cp4d_ctx *ctx, const float *ft_above) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (!ctx->have_steps || !ctx->have_data) return fail(ctx, CP4D_ESTATE, "step_dual: set_data and set_steps first");
    if (int r = check_halos(ctx, ft_above, nullptr, true, false, "step_dual: a halo slice is needed exactly on an interior face")) return r;
    if (int r = forward_into(ctx, ctx->ft, 1, ctx->sigma, ctx->g, ctx->h1)) return r;
    CK(launch_prox_f2(ctx, ctx->sigma, ctx->ft, ctx->h2, ft_above), "prox_f2");
    return CP4D_OK;
}

int cp4d_step_primal(cp4d_ctx *ctx, const float *h2z_below) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (!ctx->have_steps || !ctx->have_data) return fail(ctx, CP4D_ESTATE, "step_primal: set_data and set_steps first");
    if (int r = check_halos(ctx, nullptr, h2z_below, false, true, "step_primal: a halo slice is needed exactly on an interior face")) return r;
    if (int r = adjoint_into(ctx, ctx->h1, ctx->bp)) return r;
    CK(launch_update(ctx, ctx->tau, ctx->bp, ctx->h2, ctx->f, ctx->ft, h2z_below), "update");
    return CP4D_OK;
}

int cp4d_get_f(cp4d_ctx *ctx, float *out) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (bad_ptr(out)) return fail(ctx, CP4D_EINVAL, "get_f: bad pointer");
    CK(cudaMemcpyAsync(out, ctx->f, ctx->d.V * 4, cudaMemcpyDeviceToDevice, ctx->stream), "get_f");
    return CP4D_OK;
}

int cp4d_state_ptrs(cp4d_ctx *ctx, float **f, float **ft, float **h1, float **h2, float **g) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (f) *f = ctx->f;
    if (ft) *ft = ctx->ft;
    if (h1) *h1 = ctx->h1;
    if (h2) *h2 = ctx->h2;
    if (g) *g = ctx->g;
    return CP4D_OK;
}

int cp4d_solve_host(cp4d_ctx *ctx, const float *g_host, int32_t n_iters, float *f_host) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (ctx->z_open) return fail(ctx, CP4D_ESTATE, "solve_host: z-slab context, use the *_slab / cp4d_step_* calls");
    if (!g_host || !f_host || n_iters < 0) return fail(ctx, CP4D_EINVAL, "solve_host: bad arguments");
    if (!ctx->have_steps) return fail(ctx, CP4D_ESTATE, "solve_host: set_steps first");
    CK(cudaMemcpyAsync(ctx->g, g_host, ctx->d.S * 4, cudaMemcpyHostToDevice, ctx->stream), "solve_host h2d");
    ctx->have_data = true;
    if (int r = cp4d_reset(ctx, nullptr)) return r;
    if (int r = cp4d_iterate(ctx, n_iters)) return r;
    CK(cudaMemcpyAsync(f_host, ctx->f, ctx->d.V * 4, cudaMemcpyDeviceToHost, ctx->stream), "solve_host d2h");
    CK(cudaStreamSynchronize(ctx->stream), "solve_host sync");
    return CP4D_OK;
}

int cp4d_objective(cp4d_ctx *ctx, double *primal, double *cond_dual, double *kkt_resid) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (ctx->z_open) return fail(ctx, CP4D_ESTATE, "objective: z-slab context, use the *_slab / cp4d_step_* calls");
    if (!ctx->have_data) return fail(ctx, CP4D_ESTATE, "objective: set_data first");
    const Dims &d = ctx->d;
    double v[5] = {0, 0, 0, 0, 0};
    // primal: 1/2 |K1 f - g|^2 + lambda1 sum |K2 f|_2   (Eq. 6)
    if (int r = forward_into(ctx, ctx->f, 0, 0.f, nullptr, ctx->tmp_s)) return r;
    // |K1 f - g|^2 = |K1 f|^2 - 2 <K1 f, g> + |g|^2 with fp64-accumulated dots (products of fp32 numbers are exact in fp64)
    {
        double kk = 0, kg = 0, gg = 0;
        if (int r = cp4d_dot(ctx, ctx->tmp_s, ctx->tmp_s, (uint64_t)d.S, &kk)) return r;
        if (int r = cp4d_dot(ctx, ctx->tmp_s, ctx->g, (uint64_t)d.S, &kg)) return r;
        if (int r = cp4d_dot(ctx, ctx->g, ctx->g, (uint64_t)d.S, &gg)) return r;
        v[0] = kk - 2.0 * kg + gg;
    }
    CK(launch_tv_sum(ctx, ctx->f, ctx->red + 1), "tv");
    // dual value with the constraint K^T h = 0 ignored (G = 0): -1/2 |h1|^2 - <h1, g>; |h2| <= lambda1 holds by construction
    if (int r = cp4d_dot(ctx, ctx->h1, ctx->h1, (uint64_t)d.S, &v[2])) return r;
    if (int r = cp4d_dot(ctx, ctx->h1, ctx->g, (uint64_t)d.S, &v[3])) return r;
    // dual residual |K1^T h1 - div h2|_2 (tends to 0 at a saddle point)
    if (int r = adjoint_into(ctx, ctx->h1, ctx->bp)) return r;
    CK(launch_kkt_sum(ctx, ctx->bp, ctx->h2, ctx->red + 2), "kkt");
    double r2[2];
    CK(cudaMemcpyAsync(r2, ctx->red + 1, 2 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream), "objective copy");
    CK(cudaStreamSynchronize(ctx->stream), "objective sync");
    if (primal) *primal = 0.5 * v[0] + (double)ctx->lambda1 * r2[0];
    if (cond_dual) *cond_dual = -0.5 * v[2] - v[3];
    if (kkt_resid) *kkt_resid = std::sqrt(r2[1]);
    return CP4D_OK;
}

int cp4d_fbp(cp4d_ctx *ctx, const float *g, float *out) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    const Dims &d = ctx->d;
    const int Qf = (d.npi + 3) / 4;
    const uint64_t out_bytes = (uint64_t)d.nz * d.n * d.n * Qf * 16;
    if (bad_ptr(g) || bad_ptr(out) || overlap(g, d.S * 4, out, out_bytes)) return fail(ctx, CP4D_EINVAL, "fbp: bad pointers");
    if (Qf > d.Q) return fail(ctx, CP4D_EUNSUPPORTED, "fbp: needs ceil(n_half_rot/4)*4 <= m (the projector scratch is sized for m)");
    if ((int64_t)d.nd * 4 > 48 * 1024) return fail(ctx, CP4D_EUNSUPPORTED, "fbp: the filter keeps one sinogram row in shared memory, nd <= 12288");
    CK(launch_filter_sl(ctx, g, ctx->tmp_s), "filter");
    // the scratch rows keep their zero pads: only bins [0, nd) of the first Qf chunk planes... every plane stride is gp, and
    // with Qf != Q the row addressing differs from the fold's, so clear the scratch once and restore the invariant afterwards
    CK(cudaMemsetAsync(ctx->scratch, 0, (size_t)d.scratch4 * 16, ctx->stream), "fbp clear");
    CK(launch_fold_halfrot(ctx, ctx->tmp_s, ctx->scratch, Qf, (float)(3.14159265358979323846 / d.n0)), "fold_halfrot");
    CK(launch_backproject(ctx, ctx->scratch, out, Qf), "fbp backproject");
    CK(cudaMemsetAsync(ctx->scratch, 0, (size_t)d.scratch4 * 16, ctx->stream), "fbp clear");
    return CP4D_OK;
}

int cp4d_sync(cp4d_ctx *ctx) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    CK(cudaStreamSynchronize(ctx->stream), "sync");
    CK(cudaGetLastError(), "sync");
    return CP4D_OK;
}

int cp4d_profile_begin(cp4d_ctx *ctx) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    for (auto &r : ctx->prof) { ctx->ev_pool.push_back(r.a); ctx->ev_pool.push_back(r.b); }
    ctx->prof.clear();
    ctx->prof_on = true;
    return CP4D_OK;
}

int cp4d_profile_end(cp4d_ctx *ctx, cp4d_profile *out) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (!out) return fail(ctx, CP4D_EINVAL, "profile_end: null output");
    ctx->prof_on = false;
    std::memset(out, 0, sizeof(*out));
    CK(cudaStreamSynchronize(ctx->stream), "profile_end sync");
    for (auto &r : ctx->prof) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess && r.cls >= 0 && r.cls < CP4D_K_COUNT) {
            out->ms[r.cls] += ms;
            out->launches[r.cls]++;
        }
        ctx->ev_pool.push_back(r.a); ctx->ev_pool.push_back(r.b);
    }
    cudaGetLastError();
    ctx->prof.clear();
    return CP4D_OK;
}

const char *cp4d_kernel_name(int k) {
    static const char *names[CP4D_K_COUNT] = {"forward", "synth", "fold", "backproject", "grad", "div", "prox_f2", "update", "reduce", "misc", "mix", "prox_update"};
    return (k >= 0 && k < CP4D_K_COUNT) ? names[k] : "?";
}

int cp4d_graph_replays(const cp4d_ctx *ctx, uint64_t *out) {
    if (!ctx || !out) return CP4D_EINVAL;
    *out = ctx->graph_replays;
    return CP4D_OK;
}

int cp4d_set_projector_mode(cp4d_ctx *ctx, int32_t mode) {
    if (!ctx) return CP4D_EINVAL;
    DevGuard dev_guard(ctx->device);
    if (mode != CP4D_PROJ_AUTO && mode != CP4D_PROJ_FP32 && mode != CP4D_PROJ_TENSOR) return fail(ctx, CP4D_EINVAL, "set_projector_mode: unknown mode");
    if (mode != ctx->fw_mode) {
        if (ctx->iter_graph) {                          // the captured iteration holds the other kernels
            cudaGraphExecDestroy(ctx->iter_graph);
            ctx->iter_graph = nullptr;
        }
        // the two adjoints lay the folded sinogram out differently in the same scratch and both rely on rows whose pads are zero
        CK(cudaMemsetAsync(ctx->scratch, 0, (size_t)ctx->d.scratch4 * 16, ctx->stream), "set_projector_mode");
    }
    ctx->fw_mode = mode;
    return CP4D_OK;
}

int cp4d_projector_mode_in_use(const cp4d_ctx *ctx, int32_t *forward_out, int32_t *adjoint_out) {
    if (!ctx) return CP4D_EINVAL;
    const bool ok = forward_mma_usable(ctx);
    const bool fw_tensor = (ctx->fw_mode == CP4D_PROJ_TENSOR && ok) || (ctx->fw_mode == CP4D_PROJ_AUTO && ok && forward_mma_preferred(ctx->d));
    if (forward_out) *forward_out = fw_tensor ? CP4D_PROJ_TENSOR : CP4D_PROJ_FP32;
    if (adjoint_out) *adjoint_out = fw_tensor ? CP4D_PROJ_TENSOR : CP4D_PROJ_FP32;
    return CP4D_OK;
}

const char *cp4d_graph_note(const cp4d_ctx *ctx) { return ctx ? ctx->note.c_str() : "null context"; }

int cp4d_launch_count(const cp4d_ctx *ctx, uint64_t *out) {
    if (!ctx || !out) return CP4D_EINVAL;
    *out = ctx->launches;
    return CP4D_OK;
}

}  // extern "C"
