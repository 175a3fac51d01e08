// Forward half of the time-decomposed parallel-beam projector pair on sm_100a (Eq. 9, with the pi-fold
// of L198-L202).  A CTA stages one TILE x TILE voxel tile of one slice (all coefficients of a group) in shared memory
// once, then walks ALL base angles; every ray of the tile's window gathers its Joseph taps along the dominant axis with
// all coefficients of the group accumulated in registers, so the m coefficients are read once per tap and the synthesised
// frame sum_j Phi[j,k] f_j is never materialised.  The per-tile partial ray sums go to P[z][i][jq][b] with one vector RED
// per ray and coefficient chunk; the synthesis with Phi (and the F1* prox) is the k_synth epilogue in stream_kernels.cu.
//
//   k_forward_rays<4|2> : m % 16 == 0 (configs 3-5) / m % 8 == 0.  8 lanes per ray, voxel-major tile, conflict-free full
//                         wavefronts.
//   k_forward_partial<1>: m % 8 != 0.  One thread per ray, coefficient-plane-major tile.
//
// The backprojector lives in backproject.cu.
//
// Coordinates: the host computes, in fp64, for every (tile, base angle) the window start `bstart` and the offset
// `delta` such that the bin coordinate of tile-local voxel (lx,ly) is  u = delta + lx*c + ly*s  with 1 <= u < WIN-1;
// all fp32 arithmetic in the kernels is on these small tile-local numbers.
#include "cp4d_internal.cuh"

namespace cp4d {

constexpr int RS = TILE + 3;             // row stride of the forward tile in float4 (odd: rows rotate bank groups)
constexpr int PLANE = (TILE + 2) * RS;   // float4 per coefficient chunk plane

__device__ __forceinline__ void fma4(float4 &a, float w, const float4 &v) {
    a.x = fmaf(w, v.x, a.x); a.y = fmaf(w, v.y, a.y); a.z = fmaf(w, v.z, a.z); a.w = fmaf(w, v.w, a.w);
}

struct ProjArgs {
    int n, nz, nd, n0, Q, gp, gpl;
    const AngleTab *ang;
    const TileGeo *geo;
    const FwAngle *fwang;      // k_forward_rays: packed per-angle parameters and the angle order by stepping axis
    const int32_t *fworder;
    int n_colstep;
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


// ---------------------------------------------------------------------------------------------------
// forward, 16 or 8 coefficients per ray (m % 8 == 0): 8 lanes per ray, conflict-free shared-memory wavefronts
// ---------------------------------------------------------------------------------------------------
// The one-thread-per-ray kernel above is bound by shared-memory wavefronts, a third of which are bank conflicts (8 adjacent
// rays span up to 10 rows, rows 8 apart share a bank group) or partially filled.  Here a ray is served by 8 lanes
// = 2 step parities x 4 coefficient chunks: the tile is stored voxel-major ([row][col][16 coefficients], 64 B per voxel,
// EVEN row pitch), lane (sp, jq) handles steps k = sp, sp+2, ... and chunk jq.  The 8 lanes of a quarter warp then read two
// whole voxels, (r0, k) and (r1, k+1), whose 64 B blocks always differ in parity ((r1-r0)*pitch + 1 is odd): one full,
// conflict-free 128 B wavefront per LDS.128.  Rays that step over rows use a second pass over a transposed copy of the tile,
// so both passes run the same code.  The two step parities are summed with one shuffle before the vector RED into P.
constexpr int FR_RAYS = WIN;                 // rays of a tile window
constexpr int FR_THREADS = FR_RAYS * 8;      // 384: 8 lanes per ray
constexpr int FR_UNROLL = 4;                 // steps per lane and chunk

// JQ = coefficient chunks (float4) per voxel: 4 (16 coefficients, 64 B voxels, 2 step phases) or 2 (8 coefficients, 32 B
// voxels, 4 step phases).  Lane = (phase sp, chunk jq); the 8 lanes of a quarter warp read the voxels (r_s, k+s), s < NPH,
// whose blocks of 16*JQ bytes sit at (row*RSV + col) mod NPH = (k + s + 1) mod NPH when RSV % NPH == 0: NPH distinct
// residues, i.e. one full conflict-free 128 B wavefront per LDS.128.
template <int JQ>
struct FwRays {
    static constexpr int NPH = 8 / JQ;                          // step phases = lanes per (ray, chunk)
    static constexpr int RSV = JQ == 4 ? TILE + 2 : TILE + 4;   // voxels per tile row incl. the zero border; multiple of NPH
    static constexpr int UNROLL = FR_UNROLL;                    // steps per lane and chunk (2 and 8 were slower for JQ = 2)
    static constexpr int CHUNK = NPH * UNROLL;                  // columns of the chord per loop trip
    static constexpr size_t SMEM = (size_t)(TILE + 3) * RSV * JQ * sizeof(float4);
    static_assert(RSV % NPH == 0, "row pitch must be a multiple of the number of step phases");
};

template <int JQ>
__global__ void __launch_bounds__(FR_THREADS, 3) k_forward_rays(const float *__restrict__ f, float4 *__restrict__ P, ProjArgs a) {
    using C = FwRays<JQ>;
    constexpr int NPH = C::NPH, RSV = C::RSV, CHUNK = C::CHUNK, UNROLL = C::UNROLL;
    extern __shared__ float4 tile[];  // [TILE+3][RSV][JQ]: 1-voxel zero border, plus a second zero row at the bottom
    const int tiles_1d = (a.n + TILE - 1) / TILE;
    const int tix = blockIdx.x % tiles_1d, tiy = blockIdx.x / tiles_1d;
    const int z = blockIdx.y, jg = blockIdx.z;
    const int x0 = tix * TILE, y0 = tiy * TILE;
    const int u = threadIdx.x >> 3, sp = (threadIdx.x & 7) / JQ, jq = threadIdx.x & (JQ - 1);
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    const float4 *F = reinterpret_cast<const float4 *>(f);
    const TileGeo *geo = a.geo + (int64_t)blockIdx.x * a.n0;

    for (int t = threadIdx.x; t < (TILE + 3) * RSV * JQ; t += FR_THREADS) tile[t] = zero;   // borders stay zero in both passes
    for (int pass = 0; pass < 2; ++pass) {   // pass 0: rays stepping over columns; pass 1: over rows, on the transposed tile
        __syncthreads();
        for (int t = threadIdx.x; t < TILE * TILE * JQ; t += FR_THREADS) {
            const int jc = t & (JQ - 1), lx = (t / JQ) & (TILE - 1), ly = t / (JQ * TILE);
            const int gx = x0 + lx, gy = y0 + ly;
            const int row = pass ? lx : ly, col = pass ? ly : lx;
            tile[((row + 1) * RSV + col + 1) * JQ + jc] =
                (gx < a.n && gy < a.n) ? __ldg(F + (((int64_t)z * a.n + gy) * a.n + gx) * a.Q + jg * JQ + jc) : zero;
        }
        __syncthreads();
        const int ii0 = pass ? a.n_colstep : 0, ii1 = pass ? a.n0 : a.n_colstep;
        for (int ii = ii0; ii < ii1; ++ii) {
            const int i = a.fworder[ii];
            const FwAngle A = a.fwang[i];
            const TileGeo G = geo[i];
            // pass 0: the ray crosses column k at row (du - k c)/s; pass 1: it crosses row k at column (du - k s)/c
            const float step = A.step, base = ((float)u - G.delta) * A.inv;
            // this ray's steps k with -1 <= base + k step < TILE (one extra on each side; the body is exact on its own)
            int klo = 0, khi = TILE - 1;
            if (A.istep != 0.0f) {
                const float ta = (-1.0f - base) * A.istep, tb = ((float)TILE - base) * A.istep;
                klo = max(0, (int)floorf(fminf(ta, tb)));
                khi = min(TILE - 1, (int)ceilf(fmaxf(ta, tb)));
            } else if (!(base >= -1.0f && base < (float)TILE)) {
                klo = TILE; khi = -1;
            }
            const bool touched = klo <= khi;
            float4 acc = zero;
            // floor without the conversion pipe: tm = ys + 1.5 * 2^23 rounded DOWN holds floor(ys) in its low mantissa bits
            const float MAGIC = 12582912.0f;
            const float4 *plane = tile + jq + JQ;         // + JQ: column k lives at tile column k+1
            // per-ray chunk range: lanes of other rays in the warp are masked off, so no wavefront is spent outside the chord
            for (int kc = klo & ~(CHUNK - 1); kc <= khi; kc += CHUNK) {
                const float y0s = fmaf((float)(kc + sp), step, base);
                const float4 *pc = plane + (kc + sp) * JQ;
#pragma unroll
                for (int j = 0; j < UNROLL; ++j) {
                    const float ys = fmaf((float)(NPH * j), step, y0s);     // crossing at step k = kc + sp + NPH j
                    const float tm = __fadd_rd(ys, MAGIC);
                    const float w1 = ys - (tm - MAGIC), w0 = 1.0f - w1;     // w1 in [0,1)
                    // tile row of the first tap = floor(ys) + 1; anything outside [0, TILE] reads the two zero rows TILE+1, TILE+2
                    const unsigned row = min((unsigned)(__float_as_int(tm) - (0x4B400000 - 1)), (unsigned)(TILE + 1));
                    const float4 *p0 = reinterpret_cast<const float4 *>(reinterpret_cast<const char *>(pc) + row * (RSV * JQ * 16)) + j * (NPH * JQ);
                    const float4 v0 = p0[0], v1 = p0[RSV * JQ];
                    fma4(acc, w0, v0);
                    fma4(acc, w1, v1);
                }
            }
            // sum the step phases (lanes differing in the phase bits serve the same ray and chunk)
#pragma unroll
            for (int o = JQ; o < 8; o <<= 1) {
                acc.x += __shfl_xor_sync(0xffffffffu, acc.x, o);
                acc.y += __shfl_xor_sync(0xffffffffu, acc.y, o);
                acc.z += __shfl_xor_sync(0xffffffffu, acc.z, o);
                acc.w += __shfl_xor_sync(0xffffffffu, acc.w, o);
            }
            const int b = G.bstart + u;
            if (sp == 0 && touched && b >= 0 && b < a.nd) {
                float4 *dst = P + (((int64_t)z * a.n0 + i) * a.Q + jg * JQ + jq) * a.gp + a.gpl + b;
                atomicAdd(dst, make_float4(acc.x * A.inv_a, acc.y * A.inv_a, acc.z * A.inv_a, acc.w * A.inv_a));
            }
        }
    }
}

template <int JQ>
static cudaError_t fwd_launch_rays(cp4d_ctx *c, const float *f, float4 *P, const ProjArgs &a) {
    const Dims &d = c->d;
    const size_t sh = FwRays<JQ>::SMEM;
    cudaError_t e = cudaFuncSetAttribute(k_forward_rays<JQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh);
    if (e != cudaSuccess) return e;
    k_forward_rays<JQ><<<dim3(d.tiles, d.nz, d.Q / JQ), FR_THREADS, sh, c->stream>>>(f, P, a);
    return cudaGetLastError();
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
    ProjArgs a{d.n, d.nz, d.nd, d.n0, d.Q, d.gp, d.gpl, c->ang, c->geo, c->fwang, c->fworder, c->n_colstep};
    cudaError_t e = cudaMemsetAsync(P, 0, (size_t)d.scratch4 * sizeof(float4), c->stream);
    if (e != cudaSuccess) return e;
    c->launches += 2;
    switch (pick_jq(d.Q)) {
    case 4: return fwd_launch_rays<4>(c, f, P, a);
    case 2: return fwd_launch_rays<2>(c, f, P, a);
    default: return fwd_launch<1>(c, f, P, a);
    }
}

}  // namespace cp4d
