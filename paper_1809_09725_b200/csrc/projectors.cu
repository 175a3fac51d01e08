// Forward half of the time-decomposed parallel-beam projector pair on sm_100a (Eq. 9, with the pi-fold
// of L198-L202).  A CTA stages one TILE x TILE voxel tile (a group of coefficients of one to four slices) in shared memory
// once, then walks ALL base angles; every ray of the tile's window gathers its Joseph taps along the dominant axis with
// the coefficients accumulated in registers, so the m coefficients are read once per tap and the synthesised frame
// sum_j Phi[j,k] f_j is never materialised.  The per-tile partial ray sums go to P[z][i][b][j] (j fastest) with one vector RED
// per ray and coefficient chunk; the synthesis with Phi (and the F1* prox) is the k_synth epilogue in stream_kernels.cu.
// This is the exact-fp32 CUDA-core forward projector; forward_mma.cu holds the tensor-core one that runs by default.
//
//   k_forward_rays<JQ> : JQ = 4, 2, 1 coefficient chunks (16, 8, 4 coefficients) of 4/JQ adjacent slices per CTA.
//
// The backprojector lives in backproject.cu.
//
// Coordinates: the host computes, in fp64, for every (tile, base angle) the window start `bstart` and the offset
// `delta` such that the bin coordinate of tile-local voxel (lx,ly) is  u = delta + lx*c + ly*s  with 1 <= u < WIN-1;
// all fp32 arithmetic in the kernels is on these small tile-local numbers.
#include <algorithm>

#include "cp4d_internal.cuh"

namespace cp4d {

__device__ __forceinline__ void fma4(float4 &a, float w, const float4 &v) {
    a.x = fmaf(w, v.x, a.x); a.y = fmaf(w, v.y, a.y); a.z = fmaf(w, v.z, a.z); a.w = fmaf(w, v.w, a.w);
}

struct ProjArgs {
    int n, nz, nd, n0, Q, gp, gpl;
    const TileGeo *geo;
    const FwAngle *fwang;      // k_forward_rays: packed per-angle parameters and the angle order by stepping axis
    const int32_t *fworder;
    int n_colstep;
    int tiles, agroups;        // blockIdx.x = tile + tiles * angle group (small problems split the base angles over CTAs)
};

// ---------------------------------------------------------------------------------------------------
// forward: 8 lanes per ray, conflict-free shared-memory wavefronts
// ---------------------------------------------------------------------------------------------------
// A one-thread-per-ray gather (round 1's first kernel) is bound by shared-memory wavefronts, a third of which are bank
// conflicts (8 adjacent rays span up to 10 rows, rows 8 apart share a bank group) or partially filled.  Here a ray is served
// by 8 lanes = 2 step parities x 4 chunks of 16 B: the tile is stored voxel-major ([row][col][4 chunks], 64 B per voxel, EVEN
// row pitch), lane (sp, c4) handles steps k = sp, sp+2, ... and chunk c4.  Rays that step over rows use a second pass over a
// transposed copy of the tile, so both passes run the same code.  The two step parities are summed with one shuffle before
// the vector RED into P.
constexpr int FR_RAYS = WIN;                 // rays of a tile window
constexpr int FR_THREADS = FR_RAYS * 8;      // 384: 8 lanes per ray
constexpr int FR_UNROLL = 4;                 // steps per lane and chunk

// A shared-memory "voxel" is always 64 B = 4 float4 chunks served by 4 lanes: JQ coefficient chunks of ZZ = 4/JQ adjacent
// slices (the geometry, hence every weight, is the same for all slices).  JQ = 4: 16 coefficients of one slice; JQ = 2:
// 8 coefficients of two slices; JQ = 1: 4 coefficients of four slices.  Lane = (step parity sp, chunk c4); the 8 lanes of a
// quarter warp read the voxels (r0, k) and (r1, k+1), whose 64 B blocks differ in parity because the row pitch is even:
// one full conflict-free 128 B wavefront per LDS.128.
template <int JQ>
struct FwRays {
    static constexpr int ZZ = 4 / JQ;                           // slices per CTA
    static constexpr int NPH = 2;                               // step phases = lanes per (ray, chunk)
    static constexpr int RSV = TILE + 2;                        // voxels per tile row incl. the zero border; even
    static constexpr int UNROLL = FR_UNROLL;                    // steps per lane and chunk of the chord
    static constexpr int CHUNK = NPH * UNROLL;                  // columns of the chord per loop trip
    static constexpr size_t SMEM = (size_t)(TILE + 3) * RSV * 4 * sizeof(float4);
    static_assert(RSV % NPH == 0, "row pitch must be a multiple of the number of step phases");
};

// per-angle parameters in kernel-parameter (constant bank) space: indexed loads from it go through the constant cache, not
// through the LSU data pipe that binds this kernel.  Used when n_theta0 <= FW_TAB; otherwise the same data is read from
// global memory.
constexpr int FW_TAB = 512;
struct FwTable {
    FwAngle a[FW_TAB];
    int32_t order[FW_TAB];
};

template <int JQ, bool CONST_TAB>
__global__ void __launch_bounds__(FR_THREADS, 3) k_forward_rays(const float *__restrict__ f, float *__restrict__ P, ProjArgs a,
                                                                const __grid_constant__ FwTable tab) {
    using C = FwRays<JQ>;
    constexpr int NPH = C::NPH, RSV = C::RSV, CHUNK = C::CHUNK, UNROLL = C::UNROLL;
    constexpr int ZZ = C::ZZ;
    extern __shared__ float4 tile[];  // [TILE+3][RSV][4]: 1-voxel zero border, plus a second zero row at the bottom
    const int tiles_1d = (a.n + TILE - 1) / TILE;
    const int tile_id = blockIdx.x % a.tiles, ag = blockIdx.x / a.tiles;
    const int tix = tile_id % tiles_1d, tiy = tile_id / tiles_1d;
    const int z0 = blockIdx.y * ZZ, jg = blockIdx.z;
    const int x0 = tix * TILE, y0 = tiy * TILE;
    const int u = threadIdx.x >> 3, sp = (threadIdx.x >> 2) & 1, c4 = threadIdx.x & 3;   // chunk c4 = (slice zz, coefficient chunk jc)
    const int zz = c4 / JQ, jc = c4 % JQ, z = z0 + zz;
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    const float4 *F = reinterpret_cast<const float4 *>(f);
    const TileGeo *geo = a.geo + (int64_t)tile_id * a.n0;

    for (int t = threadIdx.x; t < (TILE + 3) * RSV * 4; t += FR_THREADS) tile[t] = zero;   // borders stay zero in both passes
    for (int pass = 0; pass < 2; ++pass) {   // pass 0: rays stepping over columns; pass 1: over rows, on the transposed tile
        // this pass's slice of the angle list, split evenly over the angle groups
        const int l0 = pass ? a.n_colstep : 0, l1 = pass ? a.n0 : a.n_colstep;
        const int ii0 = l0 + (int)((int64_t)(l1 - l0) * ag / a.agroups), ii1 = l0 + (int)((int64_t)(l1 - l0) * (ag + 1) / a.agroups);
        if (ii0 == ii1) continue;            // (CTA-uniform) no angle of this class for this CTA
        __syncthreads();
        for (int t = threadIdx.x; t < TILE * TILE * 4; t += FR_THREADS) {
            const int c = t & 3, lx = (t >> 2) & (TILE - 1), ly = t >> 7;
            const int gx = x0 + lx, gy = y0 + ly, gz = z0 + c / JQ;
            const int row = pass ? lx : ly, col = pass ? ly : lx;
            tile[((row + 1) * RSV + col + 1) * 4 + c] = (gx < a.n && gy < a.n && gz < a.nz)
                ? __ldg(F + (((int64_t)gz * a.n + gy) * a.n + gx) * a.Q + jg * JQ + c % JQ) : zero;
        }
        __syncthreads();
        for (int ii = ii0; ii < ii1; ++ii) {
            const int i = CONST_TAB ? tab.order[ii] : a.fworder[ii];
            const FwAngle A = CONST_TAB ? tab.a[i] : a.fwang[i];
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
            const float4 *plane = tile + c4 + 4;          // + 4: column k lives at tile column k+1
            // per-ray chunk range: lanes of other rays in the warp are masked off, so no wavefront is spent outside the chord
            for (int kc = klo & ~(CHUNK - 1); kc <= khi; kc += CHUNK) {
                const float y0s = fmaf((float)(kc + sp), step, base);
                const float4 *pc = plane + (kc + sp) * 4;
#pragma unroll
                for (int j = 0; j < UNROLL; ++j) {
                    const float ys = fmaf((float)(NPH * j), step, y0s);     // crossing at step k = kc + sp + NPH j
                    const float tm = __fadd_rd(ys, MAGIC);
                    const float w1 = ys - (tm - MAGIC), w0 = 1.0f - w1;     // w1 in [0,1)
                    // tile row of the first tap = floor(ys) + 1; anything outside [0, TILE] reads the two zero rows TILE+1, TILE+2
                    const unsigned row = min((unsigned)(__float_as_int(tm) - (0x4B400000 - 1)), (unsigned)(TILE + 1));
                    const float4 *p0 = reinterpret_cast<const float4 *>(reinterpret_cast<const char *>(pc) + row * (RSV * 64)) + j * (NPH * 4);
                    const float4 v0 = p0[0], v1 = p0[RSV * 4];
                    fma4(acc, w0, v0);
                    fma4(acc, w1, v1);
                }
            }
            // sum the two step parities (lanes l and l^4 serve the same ray and chunk) with 2 shuffles instead of 4: the sp = 0
            // lane ends up with the (x, y) totals, the sp = 1 lane with (z, w), and each adds its half to P with one 8-byte RED
            const float s0 = sp ? acc.x : acc.z, s1 = sp ? acc.y : acc.w;          // what the partner needs
            const float r0 = __shfl_xor_sync(0xffffffffu, s0, 4), r1 = __shfl_xor_sync(0xffffffffu, s1, 4);
            const float2 tot = sp ? make_float2(acc.z + r0, acc.w + r1) : make_float2(acc.x + r0, acc.y + r1);
            const int b = G.bstart + u;
            if (touched && b >= 0 && b < a.nd && z < a.nz) {
                float2 *dst = reinterpret_cast<float2 *>(P + ((((int64_t)z * a.n0 + i) * a.gp + a.gpl + b) * a.Q + jg * JQ + jc) * 4) + sp;
                atomicAdd(dst, make_float2(tot.x, tot.y));          // 1/a is applied by k_synth
            }
        }
    }
}

template <int JQ>
static cudaError_t fwd_launch_rays(cp4d_ctx *c, const float *f, float *P, const ProjArgs &a) {
    const Dims &d = c->d;
    const size_t sh = FwRays<JQ>::SMEM;
    // small problems: split the base angles over up to 8 CTAs per tile
    const int nzz = (a.nz + FwRays<JQ>::ZZ - 1) / FwRays<JQ>::ZZ;
    const int64_t ctas = (int64_t)d.tiles * nzz * (d.Q / JQ);
    ProjArgs b = a;
    // whole waves of 148 SMs x 3 resident CTAs: pick the split with the least (waves x work per CTA), the work of a CTA being its
    // share of the base angles plus the staging of its tile and its REDs (about 16 angles' worth, measured)
    b.agroups = 1;
    double best = 1e300;
    for (int ag = 1; ag <= std::min(8, d.n0); ++ag) {
        const int64_t waves = (ctas * ag + 148 * 3 - 1) / (148 * 3);
        const double cost = (double)waves * ((d.n0 + ag - 1) / ag + 16);
        if (cost < best) { best = cost; b.agroups = ag; }
    }
    const dim3 grid(d.tiles * b.agroups, nzz, d.Q / JQ);
    if (d.n0 <= FW_TAB)
        k_forward_rays<JQ, true><<<grid, FR_THREADS, sh, c->stream>>>(f, P, b, *c->fwtab_host);
    else
        k_forward_rays<JQ, false><<<grid, FR_THREADS, sh, c->stream>>>(f, P, b, FwTable{});
    return cudaGetLastError();
}

template <int JQ>
static cudaError_t fwd_init_one() {
    cudaError_t e = cudaFuncSetAttribute(k_forward_rays<JQ, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FwRays<JQ>::SMEM);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_forward_rays<JQ, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FwRays<JQ>::SMEM);
}
// cp4d_create calls this once per context (the attribute is per device and sticks)
cudaError_t forward_init() {
    cudaError_t e;
    if ((e = fwd_init_one<4>()) != cudaSuccess || (e = fwd_init_one<2>()) != cudaSuccess || (e = fwd_init_one<1>()) != cudaSuccess) return e;
    return forward_mma_init();
}

static int pick_jq(int Q) { return (Q % 4 == 0) ? 4 : (Q % 2 == 0) ? 2 : 1; }

FwTable *fwtable_new(const FwAngle *ang, const int32_t *order, int n0) {
    if (n0 > FW_TAB) return nullptr;
    FwTable *t = new FwTable();
    for (int i = 0; i < n0; ++i) { t->a[i] = ang[i]; t->order[i] = order[i]; }
    return t;
}
void fwtable_free(FwTable *t) { delete t; }

cudaError_t launch_forward_partial(cp4d_ctx *c, const float *f, float4 *P) {
    ProfScope ps(c, CP4D_K_FORWARD);
    const Dims &d = c->d;
    ProjArgs a{d.n, d.nz, d.nd, d.n0, d.Q, d.nd, 0, c->geo, c->fwang, c->fworder, c->n_colstep, d.tiles, 1};
    cudaError_t e = cudaMemsetAsync(P, 0, (size_t)d.nz * d.n0 * d.nd * d.Q * sizeof(float4), c->stream);
    if (e != cudaSuccess) return e;
    c->launches += 2;
    float *Pf = reinterpret_cast<float *>(P);
    if (forward_mma_usable(c) && (c->fw_mode == CP4D_PROJ_TENSOR || (c->fw_mode == CP4D_PROJ_AUTO && forward_mma_preferred(d))))
        return launch_forward_mma(c, f, Pf);
    switch (pick_jq(d.Q)) {
    case 4: return fwd_launch_rays<4>(c, f, Pf, a);
    case 2: return fwd_launch_rays<2>(c, f, Pf, a);
    default: return fwd_launch_rays<1>(c, f, Pf, a);
    }
}

}  // namespace cp4d
