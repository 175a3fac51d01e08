// The fused streaming step of the CP iteration (Fig. 2, steps 4-6 in one pass):
//     h2+ = proj_{|.| <= lambda1}(h2 + sigma K2 ft)                          (step 4)
//     f+  = f - tau K1^T h1 + tau div h2+ ;  ft+ = f+ + theta (f+ - f)      (steps 5-6)
// k_grad<1> + k_div<1> (stream_kernels.cu) move 9 V + 8 V floats through HBM; here h2+ goes from the prox to the divergence
// through shared memory, so an iteration reads ft, h2[4], K1^T h1, f and writes h2+[4], f+, ft+: 13 V.
//
// The divergence at a voxel needs h2+ at its x-1, y-1, z-1 and t-1 neighbours.  A CTA owns a tile of FU_TX x ty voxels (all
// 4D coefficients of them) and walks along z: it computes the prox also on the one-voxel halo column x0-1 and halo row y0-1
// (the neighbour CTA computes the same values with the same instructions), keeps the z-1 slice of h2z+ in shared memory, and
// synchronises between the prox and the update of a slice.  Because a neighbour CTA recomputes the prox on my border voxels
// from the OLD h2 and ft at a time I do not control, h2+ and ft+ go to second copies of the two arrays (h2_new, ft_new); the
// host swaps the roles after every pass.  f and K1^T h1 are read and written by the owner of the voxel only: in place.
// A z-chunk that does not start at slice 0 first recomputes h2z+ of the slice below it (prox only, nothing stored).
//
// The arithmetic is that of k_grad<1> and k_div<1>, expression by expression, so both paths give the same iterates.
#include <algorithm>

#include "cp4d_internal.cuh"

namespace cp4d {

namespace {

constexpr int FU_TX = 16;            // tile width in voxels; the height ty follows from Q (launcher)
constexpr int FU_THREADS = 256;
constexpr int FU_BAND = 8;            // tile rows per band of the launch order
constexpr int FU_KMAX = 2;           // elements per thread: (FU_TX + 1) * (ty + 1) * Q <= FU_KMAX * FU_THREADS
constexpr int FU_SMEM_MAX = 5 * FU_KMAX * FU_THREADS * 16;

struct FusedArgs {
    int n, nz, Q, zper, ty, tiles_x, tiles_y, l1_zero;
    int slice4;                      // float4 per slice (< 2^31: validate() bounds n * n * Q)
    int64_t V4;
    float lambda2, sigma, inv_l1, tau, theta;
};

enum : unsigned { FL_LIVE = 1, FL_OWN = 2, FL_XP = 4, FL_YP = 8, FL_TP = 16, FL_XM = 32, FL_YM = 64, FL_TM = 128 };

__device__ __forceinline__ float4 ldg4(const float4 *p) { return __ldg(p); }
__device__ __forceinline__ float4 diff4(float4 a, float4 b) { return make_float4(a.x - b.x, a.y - b.y, a.z - b.z, a.w - b.w); }

__global__ void __launch_bounds__(FU_THREADS, 4) k_prox_update(const float4 *__restrict__ ft, const float4 *__restrict__ h2,
                                                            float4 *__restrict__ h2n, const float4 *__restrict__ bp,
                                                            float4 *f, float4 *__restrict__ ftn, FusedArgs a) {
    extern __shared__ float4 fu_sm[];
    const int W = (FU_TX + 1) * a.Q, items = W * (a.ty + 1);
    float4 *s_hx = fu_sm, *s_hy = fu_sm + items, *s_ht = fu_sm + 2 * items, *s_hz = fu_sm + 3 * items;      // s_hz: two slices
    // tiles in bands of FU_BAND tile rows, inside a band column by column: CTAs next to each other in launch order share a halo
    // row and walk z in step, so the halo reads of one are the other's own reads of a moment ago (L2 hits at any N)
    const int per_band = a.tiles_x * FU_BAND, band = blockIdx.x / per_band, rb = blockIdx.x - band * per_band;
    const int rows = min(FU_BAND, a.tiles_y - band * FU_BAND);
    const int x0 = (rb / rows) * FU_TX, y0 = (band * FU_BAND + rb % rows) * a.ty;
    const int z0 = blockIdx.y * a.zper, z1 = min(a.nz, z0 + a.zper);
    const int sy = a.n * a.Q;

    // my elements of the extended tile (ey, ex, c), c fastest: ex = 0 is the halo column x0 - 1, ey = 0 the halo row y0 - 1
    int goff[FU_KMAX];               // float4 offset inside a slice
    unsigned flag[FU_KMAX];
#pragma unroll
    for (int k = 0; k < FU_KMAX; ++k) {
        const int e = threadIdx.x + k * FU_THREADS;
        const int c = e % a.Q, ex = (e / a.Q) % (FU_TX + 1), ey = e / W;
        const int x = x0 - 1 + ex, y = y0 - 1 + ey;
        unsigned fl = 0;
        if (e < items && x >= 0 && y >= 0 && x < a.n && y < a.n) {
            fl = FL_LIVE;
            if (ex > 0 && ey > 0) fl |= FL_OWN;
            if (x + 1 < a.n) fl |= FL_XP;
            if (y + 1 < a.n) fl |= FL_YP;
            if (c + 1 < a.Q) fl |= FL_TP;
            if (x > 0) fl |= FL_XM;
            if (y > 0) fl |= FL_YM;
            if (c > 0) fl |= FL_TM;
        }
        flag[k] = fl;
        goff[k] = fl ? (y * a.n + x) * a.Q + c : 0;      // (a dead element loads from offset 0 and stores nothing)
    }
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);

    for (int z = z0 > 0 ? z0 - 1 : z0; z < z1; ++z) {
        const bool pre = z < z0;     // the slice below the chunk: only h2z+ of my own voxels is needed
        float4 *hz_cur = s_hz + (z & 1) * items;
        const float4 *hz_prev = s_hz + ((z & 1) ^ 1) * items;
        // ---- step 4 on the extended tile ----
#pragma unroll
        for (int k = 0; k < FU_KMAX; ++k) {
            const unsigned fl = flag[k];
            // no branches around the loads, so that those of all my elements are in flight together: a missing neighbour
            // is the element itself (difference 0), a dead element computes on offset 0 and stores nothing
            const bool act = (fl & FL_LIVE) && !(pre && !(fl & FL_OWN));
            const int e = threadIdx.x + k * FU_THREADS;
            const int64_t idx = (int64_t)z * a.slice4 + goff[k];
            const float4 cur = ldg4(ft + idx);
            const float4 fz = ldg4(ft + idx + ((z + 1 < a.nz) ? a.slice4 : 0));
            const float4 fx = ldg4(ft + idx + ((fl & FL_XP) ? a.Q : 0));
            const float4 fy = ldg4(ft + idx + ((fl & FL_YP) ? sy : 0));
            const float ftp = __ldg(reinterpret_cast<const float *>(ft) + idx * 4 + ((fl & FL_TP) ? 4 : 3));
            const float4 qx = ldg4(h2 + idx), qy = ldg4(h2 + idx + a.V4), qz = ldg4(h2 + idx + 2 * a.V4), qt = ldg4(h2 + idx + 3 * a.V4);
            float4 gx = diff4(fx, cur), gy = diff4(fy, cur), gz = diff4(fz, cur);
            float4 gt = make_float4(a.lambda2 * (cur.y - cur.x), a.lambda2 * (cur.z - cur.y), a.lambda2 * (cur.w - cur.z),
                                    a.lambda2 * (ftp - cur.w));
#define CP4D_FU_PROX(C)                                                                                       \
    {                                                                                                         \
        float vx = fmaf(a.sigma, gx.C, qx.C), vy = fmaf(a.sigma, gy.C, qy.C), vz = fmaf(a.sigma, gz.C, qz.C), \
              vt = fmaf(a.sigma, gt.C, qt.C);                                                                 \
        float nn = sqrtf(fmaf(vx, vx, fmaf(vy, vy, fmaf(vz, vz, vt * vt))));                                  \
        float r = a.l1_zero ? 0.0f : 1.0f / fmaxf(1.0f, nn * a.inv_l1);                                       \
        gx.C = vx * r; gy.C = vy * r; gz.C = vz * r; gt.C = vt * r;                                           \
    }
            CP4D_FU_PROX(x) CP4D_FU_PROX(y) CP4D_FU_PROX(z) CP4D_FU_PROX(w)
#undef CP4D_FU_PROX
            if (act) hz_cur[e] = gz;
            if (act && !pre) {
                s_hx[e] = gx; s_hy[e] = gy; s_ht[e] = gt;
                if (fl & FL_OWN) {
                    h2n[idx] = gx; h2n[idx + a.V4] = gy; h2n[idx + 2 * a.V4] = gz; h2n[idx + 3 * a.V4] = gt;
                }
            }
        }
        // f and K1^T h1 of my own voxels: on their way while the CTA meets at the barrier
        float4 fo_k[FU_KMAX], b_k[FU_KMAX];
#pragma unroll
        for (int k = 0; k < FU_KMAX; ++k) {
            // (elements I do not own read offset 0 of the slice and use nothing of it)
            const int64_t idx = (int64_t)z * a.slice4 + ((flag[k] & FL_OWN) ? goff[k] : 0);
            fo_k[k] = f[idx];
            b_k[k] = ldg4(bp + idx);
        }
        __syncthreads();
        // ---- steps 5-6 on my own voxels ----
        if (!pre) {
#pragma unroll
            for (int k = 0; k < FU_KMAX; ++k) {
                const unsigned fl = flag[k];
                if (!(fl & FL_OWN)) continue;
                const int e = threadIdx.x + k * FU_THREADS;
                const int64_t idx = (int64_t)z * a.slice4 + goff[k];
                const float4 xc = (fl & FL_XP) ? s_hx[e] : zero;
                const float4 xm = (fl & FL_XM) ? s_hx[e - a.Q] : zero;
                const float4 yc = (fl & FL_YP) ? s_hy[e] : zero;
                const float4 ym = (fl & FL_YM) ? s_hy[e - W] : zero;
                const float4 zc = (z < a.nz - 1) ? hz_cur[e] : zero;
                const float4 prevz = (z > 0) ? hz_prev[e] : zero;
                const float4 tc = s_ht[e];
                const float tm = (fl & FL_TM) ? s_ht[e - 1].w : 0.0f;
                const float tw = (fl & FL_TP) ? tc.w : 0.0f;
                float4 d;
                d.x = (xc.x - xm.x) + (yc.x - ym.x) + (zc.x - prevz.x) + a.lambda2 * (tc.x - tm);
                d.y = (xc.y - xm.y) + (yc.y - ym.y) + (zc.y - prevz.y) + a.lambda2 * (tc.y - tc.x);
                d.z = (xc.z - xm.z) + (yc.z - ym.z) + (zc.z - prevz.z) + a.lambda2 * (tc.z - tc.y);
                d.w = (xc.w - xm.w) + (yc.w - ym.w) + (zc.w - prevz.w) + a.lambda2 * (tw - tc.z);
                const float4 fo = fo_k[k], b = b_k[k];
                float4 fn, fr;
                fn.x = fmaf(a.tau, d.x - b.x, fo.x); fn.y = fmaf(a.tau, d.y - b.y, fo.y);
                fn.z = fmaf(a.tau, d.z - b.z, fo.z); fn.w = fmaf(a.tau, d.w - b.w, fo.w);
                fr.x = fmaf(a.theta, fn.x - fo.x, fn.x); fr.y = fmaf(a.theta, fn.y - fo.y, fn.y);
                fr.z = fmaf(a.theta, fn.z - fo.z, fn.z); fr.w = fmaf(a.theta, fn.w - fo.w, fn.w);
                f[idx] = fn;
                ftn[idx] = fr;
            }
            __syncthreads();         // the next slice's prox overwrites s_hx, s_hy, s_ht (and the older s_hz slice)
        }
    }
}

}  // namespace

cudaError_t fused_step_init() {
    return cudaFuncSetAttribute(k_prox_update, cudaFuncAttributeMaxDynamicSharedMemorySize, FU_SMEM_MAX);
}

// h2_new, ft_new: the second copies (same sizes as h2, ft); on return the caller swaps (h2, h2_new) and (ft, ft_new)
cudaError_t launch_prox_update(cp4d_ctx *c, float sigma, float tau, const float *ft, const float *h2, float *h2_new,
                               const float *bp, float *f, float *ft_new) {
    ProfScope ps(c, CP4D_K_PROX_UPDATE);
    const Dims &d = c->d;
    FusedArgs a;
    a.n = d.n; a.nz = d.nz; a.Q = d.Qp; a.slice4 = (int)d.slice4; a.V4 = (int64_t)(d.V / 4);
    a.lambda2 = c->lambda2; a.sigma = sigma; a.tau = tau; a.theta = c->theta;
    a.l1_zero = !(c->lambda1 > 0.f); a.inv_l1 = a.l1_zero ? 0.f : 1.0f / c->lambda1;
    a.ty = std::max(1, 32 / a.Q);
    while (a.ty > 1 && (FU_TX + 1) * (a.ty + 1) * a.Q > FU_KMAX * FU_THREADS) --a.ty;
    const int items = (FU_TX + 1) * (a.ty + 1) * a.Q;
    if (items > FU_KMAX * FU_THREADS) return cudaErrorInvalidConfiguration;
    a.tiles_x = (d.n + FU_TX - 1) / FU_TX;
    a.tiles_y = (d.n + a.ty - 1) / a.ty;
    const int64_t tiles = (int64_t)a.tiles_x * a.tiles_y;
    // enough CTAs to fill the GPU a few times over; otherwise split z (each chunk recomputes the prox of one slice below it)
    int zchunks = 1;
    while (tiles * zchunks < 148 * 8 && zchunks * 4 <= d.nz) zchunks *= 2;
    a.zper = (d.nz + zchunks - 1) / zchunks;
    const dim3 grid((unsigned)tiles, (unsigned)((d.nz + a.zper - 1) / a.zper));
    k_prox_update<<<grid, FU_THREADS, (size_t)5 * items * sizeof(float4), c->stream>>>(
        reinterpret_cast<const float4 *>(ft), reinterpret_cast<const float4 *>(h2), reinterpret_cast<float4 *>(h2_new),
        reinterpret_cast<const float4 *>(bp), reinterpret_cast<float4 *>(f), reinterpret_cast<float4 *>(ft_new), a);
    c->launches++;
    return cudaGetLastError();
}

}  // namespace cp4d
