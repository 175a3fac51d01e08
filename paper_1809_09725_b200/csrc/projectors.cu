// Time-decomposed parallel-beam projector pair on sm_100a (Eq. 9/10, L184/L196, with the pi-fold of
// L198-L212).  Both kernels work on TILE x TILE voxel tiles of one slice and keep all coefficients j of a
// ray / voxel in registers, so the m coefficients are read once per tap and the synthesised frame
// sum_j Phi[j,k] f_j is never materialised:
//
//   k_forward_partial : the CTA stages its f tile (all j of a chunk group) in shared memory once, then walks ALL
//                       base angles; a thread owns one ray (bin) of the tile's window at that angle and gathers the
//                       Joseph taps along the dominant axis (2 LDS.128 + 8 FFMA per step and coefficient chunk);
//                       the per-tile partial ray sums go to P[z][i][jc][b] with one vector RED per ray and chunk.
//                       The synthesis with Phi (and the F1* prox) is the k_synth epilogue in stream_kernels.cu.
//   k_backproject     : voxel-driven gather from the folded sinogram gt[z][i][jc][b]; the <= WIN bins a tile can touch
//                       at an angle are staged in shared memory with cp.async (zero-fill outside the detector),
//                       double-buffered over chunks of ANG_CHUNK angles; a thread owns 4 voxels x all j of the group.
//
// Coordinates: the host computes, in fp64, for every (tile, base angle) the window start `bstart` and the offset
// `delta` such that the bin coordinate of tile-local voxel (lx,ly) is  u = delta + lx*c + ly*s  with 1 <= u < WIN-1;
// all fp32 arithmetic in the kernels is on these small tile-local numbers.
#include "cp4d_internal.cuh"

namespace cp4d {

constexpr int ANG_CHUNK = 8;
constexpr int RS = TILE + 3;             // row stride of the forward tile in float4 (odd: rows rotate bank groups)
constexpr int PLANE = (TILE + 2) * RS;   // float4 per coefficient chunk plane

__device__ __forceinline__ void fma4(float4 &a, float w, const float4 &v) {
    a.x = fmaf(w, v.x, a.x); a.y = fmaf(w, v.y, a.y); a.z = fmaf(w, v.z, a.z); a.w = fmaf(w, v.w, a.w);
}

struct ProjArgs {
    int n, nz, nd, n0, Q;
    const AngleTab *ang;
    const TileGeo *geo;
};

// ---------------------------------------------------------------------------------------------------
// forward: partial ray sums of one tile for all base angles
// ---------------------------------------------------------------------------------------------------
template <int JQ>
__global__ void __launch_bounds__(256) k_forward_partial(const float *__restrict__ f, float4 *__restrict__ P, ProjArgs a) {
    extern __shared__ float4 tile[];  // [JQ][TILE+2][RS], 1-cell zero border
    const int tiles_1d = (a.n + TILE - 1) / TILE;
    const int tix = blockIdx.x % tiles_1d, tiy = blockIdx.x / tiles_1d;
    const int z = blockIdx.y, jg = blockIdx.z;
    const int x0 = tix * TILE, y0 = tiy * TILE;
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int t = threadIdx.x; t < JQ * PLANE; t += blockDim.x) tile[t] = zero;
    __syncthreads();
    const float4 *F = reinterpret_cast<const float4 *>(f);
    for (int t = threadIdx.x; t < TILE * TILE * JQ; t += blockDim.x) {
        const int jc = t % JQ, lx = (t / JQ) % TILE, ly = t / (JQ * TILE);
        const int gx = x0 + lx, gy = y0 + ly;
        if (gx < a.n && gy < a.n)
            tile[jc * PLANE + (ly + 1) * RS + lx + 1] = __ldg(F + (((int64_t)z * a.n + gy) * a.n + gx) * a.Q + jg * JQ + jc);
    }
    __syncthreads();

    const int slot = threadIdx.x >> 6, u = threadIdx.x & 63;
    if (u >= WIN) return;
    const TileGeo *geo = a.geo + (int64_t)blockIdx.x * a.n0;
    for (int i = slot; i < a.n0; i += 4) {
        const TileGeo G = geo[i];
        const AngleTab A = a.ang[i];
        float4 acc[JQ];
#pragma unroll
        for (int jc = 0; jc < JQ; ++jc) acc[jc] = zero;
        bool touched = false;
        const float du = (float)u - G.delta;
        if (A.col_step) {
            // ray crosses column lx at local row (du - lx c)/s ; taps rows r, r+1
            const float inv = 1.0f / A.s, step = -A.c * inv, base = du * inv;
#pragma unroll 4
            for (int lx = 0; lx < TILE; ++lx) {
                const float ys = fmaf((float)lx, step, base);
                const float fl = floorf(ys);
                const int r = (int)fl;
                if ((unsigned)(r + 1) <= (unsigned)TILE) {
                    const float w1 = ys - fl, w0 = 1.0f - w1;
                    const float4 *p0 = tile + (r + 1) * RS + lx + 1;
#pragma unroll
                    for (int jc = 0; jc < JQ; ++jc) {
                        const float4 t0 = p0[jc * PLANE], t1 = p0[jc * PLANE + RS];
                        fma4(acc[jc], w0, t0);
                        fma4(acc[jc], w1, t1);
                    }
                    touched = true;
                }
            }
        } else {
            const float inv = 1.0f / A.c, step = -A.s * inv, base = du * inv;
#pragma unroll 4
            for (int ly = 0; ly < TILE; ++ly) {
                const float xs = fmaf((float)ly, step, base);
                const float fl = floorf(xs);
                const int q = (int)fl;
                if ((unsigned)(q + 1) <= (unsigned)TILE) {
                    const float w1 = xs - fl, w0 = 1.0f - w1;
                    const float4 *p0 = tile + (ly + 1) * RS + q + 1;
#pragma unroll
                    for (int jc = 0; jc < JQ; ++jc) {
                        const float4 t0 = p0[jc * PLANE], t1 = p0[jc * PLANE + 1];
                        fma4(acc[jc], w0, t0);
                        fma4(acc[jc], w1, t1);
                    }
                    touched = true;
                }
            }
        }
        const int b = G.bstart + u;
        if (touched && b >= 0 && b < a.nd) {
            float4 *dst = P + (((int64_t)z * a.n0 + i) * a.Q + jg * JQ) * a.nd + b;
#pragma unroll
            for (int jc = 0; jc < JQ; ++jc) {
                const float4 v = make_float4(acc[jc].x * A.inv_a, acc[jc].y * A.inv_a, acc[jc].z * A.inv_a, acc[jc].w * A.inv_a);
                atomicAdd(dst + (int64_t)jc * a.nd, v);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// adjoint: backprojection of the folded sinogram over the base angles
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem, int src_bytes) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(sa), "l"(gmem), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

template <int JQ>
__global__ void __launch_bounds__(256, 2) k_backproject(const float4 *__restrict__ gt, float *__restrict__ out, ProjArgs a) {
    extern __shared__ float4 smem_bp[];
    float4(*win)[ANG_CHUNK][JQ][WIN] = reinterpret_cast<float4(*)[ANG_CHUNK][JQ][WIN]>(smem_bp);
    float4(*sgeo)[ANG_CHUNK] = reinterpret_cast<float4(*)[ANG_CHUNK]>(smem_bp + 2 * ANG_CHUNK * JQ * WIN);  // delta, c, s, inv_a
    const int tiles_1d = (a.n + TILE - 1) / TILE;
    const int tix = blockIdx.x % tiles_1d, tiy = blockIdx.x / tiles_1d;
    const int z = blockIdx.y, jg = blockIdx.z;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const TileGeo *geo = a.geo + (int64_t)blockIdx.x * a.n0;
    const int nch = (a.n0 + ANG_CHUNK - 1) / ANG_CHUNK;

    auto stage = [&](int buf, int ch) {
        const int i0 = ch * ANG_CHUNK;
        if (threadIdx.x < ANG_CHUNK) {
            const int i = i0 + threadIdx.x;
            float4 g4 = make_float4(1.f, 0.f, 0.f, 0.f);
            if (i < a.n0) {
                const AngleTab A = a.ang[i];
                g4 = make_float4(geo[i].delta, A.c, A.s, A.inv_a);
            }
            sgeo[buf][threadIdx.x] = g4;
        }
        for (int t = threadIdx.x; t < ANG_CHUNK * JQ * WIN; t += blockDim.x) {
            const int w = t % WIN, jc = (t / WIN) % JQ, aa = t / (WIN * JQ);
            const int i = i0 + aa;
            bool ok = i < a.n0;
            int b = 0;
            if (ok) { b = geo[i].bstart + w; ok = (b >= 0) && (b < a.nd); }
            const float4 *src = ok ? gt + (((int64_t)z * a.n0 + i) * a.Q + jg * JQ + jc) * a.nd + b : gt;
            cp_async16(&win[buf][aa][jc][w], src, ok ? 16 : 0);
        }
        cp_async_commit();
    };

    float4 acc[4][JQ];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int jc = 0; jc < JQ; ++jc) acc[r][jc] = make_float4(0.f, 0.f, 0.f, 0.f);

    stage(0, 0);
    for (int ch = 0; ch < nch; ++ch) {
        const int buf = ch & 1;
        if (ch + 1 < nch) { stage(buf ^ 1, ch + 1); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        __syncthreads();
        const int na = min(ANG_CHUNK, a.n0 - ch * ANG_CHUNK);
        for (int aa = 0; aa < na; ++aa) {
            const float4 G = sgeo[buf][aa];
            const float u0 = fmaf((float)tx, G.y, fmaf((float)ty, G.z, G.x));
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const float uu = fmaf((float)(8 * r), G.z, u0);
                const float fl = floorf(uu);
                const float fr = uu - fl;
                const float w0 = fmaxf(0.f, 1.0f - fr * G.w) * G.w;
                const float w1 = fmaxf(0.f, 1.0f - (1.0f - fr) * G.w) * G.w;
                const float4 *wp = &win[buf][aa][0][(int)fl];
#pragma unroll
                for (int jc = 0; jc < JQ; ++jc) {
                    const float4 t0 = wp[jc * WIN], t1 = wp[jc * WIN + 1];
                    fma4(acc[r][jc], w0, t0);
                    fma4(acc[r][jc], w1, t1);
                }
            }
        }
        __syncthreads();
    }
    float4 *O = reinterpret_cast<float4 *>(out);
    const int x = tix * TILE + tx;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int y = tiy * TILE + ty + 8 * r;
        if (x < a.n && y < a.n) {
            float4 *dst = O + (((int64_t)z * a.n + y) * a.n + x) * a.Q + jg * JQ;
#pragma unroll
            for (int jc = 0; jc < JQ; ++jc) dst[jc] = acc[r][jc];
        }
    }
}

static int pick_jq(int Q) { return (Q % 4 == 0) ? 4 : (Q % 2 == 0) ? 2 : 1; }

template <int JQ>
static cudaError_t fwd_launch(cp4d_ctx *c, const float *f, float4 *P, const ProjArgs &a) {
    const Dims &d = c->d;
    const size_t sh = (size_t)JQ * PLANE * sizeof(float4);
    cudaError_t e = cudaFuncSetAttribute(k_forward_partial<JQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh);
    if (e != cudaSuccess) return e;
    k_forward_partial<JQ><<<dim3(d.tiles, d.nz, d.Q / JQ), 256, sh, c->stream>>>(f, P, a);
    return cudaGetLastError();
}

template <int JQ>
static cudaError_t bp_launch(cp4d_ctx *c, const float4 *gt, float *f_out, const ProjArgs &a) {
    const Dims &d = c->d;
    const size_t sh = (size_t)(2 * ANG_CHUNK * JQ * WIN + 2 * ANG_CHUNK) * sizeof(float4);
    cudaError_t e = cudaFuncSetAttribute(k_backproject<JQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh);
    if (e != cudaSuccess) return e;
    k_backproject<JQ><<<dim3(d.tiles, d.nz, d.Q / JQ), 256, sh, c->stream>>>(gt, f_out, a);
    return cudaGetLastError();
}

cudaError_t launch_forward_partial(cp4d_ctx *c, const float *f, float4 *P) {
    ProfScope ps(c, CP4D_K_FORWARD);
    const Dims &d = c->d;
    ProjArgs a{d.n, d.nz, d.nd, d.n0, d.Q, c->ang, c->geo};
    cudaError_t e = cudaMemsetAsync(P, 0, (size_t)d.scratch4 * sizeof(float4), c->stream);
    if (e != cudaSuccess) return e;
    c->launches += 2;
    switch (pick_jq(d.Q)) {
    case 4: return fwd_launch<4>(c, f, P, a);
    case 2: return fwd_launch<2>(c, f, P, a);
    default: return fwd_launch<1>(c, f, P, a);
    }
}

cudaError_t launch_backproject(cp4d_ctx *c, const float4 *gt, float *f_out) {
    ProfScope ps(c, CP4D_K_BACKPROJECT);
    const Dims &d = c->d;
    ProjArgs a{d.n, d.nz, d.nd, d.n0, d.Q, c->ang, c->geo};
    c->launches++;
    switch (pick_jq(d.Q)) {
    case 4: return bp_launch<4>(c, gt, f_out, a);
    case 2: return bp_launch<2>(c, gt, f_out, a);
    default: return bp_launch<1>(c, gt, f_out, a);
    }
}

}  // namespace cp4d
