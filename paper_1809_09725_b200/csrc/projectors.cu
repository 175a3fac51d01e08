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
    int n, nz, nd, n0, Q, gp, gpl;
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
            float4 *dst = P + (((int64_t)z * a.n0 + i) * a.Q + jg * JQ) * a.gp + a.gpl + b;
#pragma unroll
            for (int jc = 0; jc < JQ; ++jc) {
                const float4 v = make_float4(acc[jc].x * A.inv_a, acc[jc].y * A.inv_a, acc[jc].z * A.inv_a, acc[jc].w * A.inv_a);
                atomicAdd(dst + (int64_t)jc * a.gp, v);
            }
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

cudaError_t launch_forward_partial(cp4d_ctx *c, const float *f, float4 *P) {
    ProfScope ps(c, CP4D_K_FORWARD);
    const Dims &d = c->d;
    ProjArgs a{d.n, d.nz, d.nd, d.n0, d.Q, d.gp, d.gpl, c->ang, c->geo};
    cudaError_t e = cudaMemsetAsync(P, 0, (size_t)d.scratch4 * sizeof(float4), c->stream);
    if (e != cudaSuccess) return e;
    c->launches += 2;
    switch (pick_jq(d.Q)) {
    case 4: return fwd_launch<4>(c, f, P, a);
    case 2: return fwd_launch<2>(c, f, P, a);
    default: return fwd_launch<1>(c, f, P, a);
    }
}

}  // namespace cp4d
