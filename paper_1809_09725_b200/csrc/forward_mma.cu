// Forward projector on the tensor cores (Eq. 9, with the pi-fold of L198-L202): the Joseph ray sums of all
// coefficients over the base angles, as small products  D[16 rays x 8 batch entries] += W[16 rays x 32 voxels] * F[32 voxels x 8]
// with the weight block W as the 2:4 SPARSE operand of mma.sp (SASS HMMA.SP.16832).
//
// Why.  The CUDA-core gather (projectors.cu) needs one shared-memory word per FMA and sits on the LSU data pipe at 0.19 of
// the FP32 peak.  The interpolation weights do not depend on the slice or on the coefficient, so the batch axis (slice, j) is
// a dense axis: a block of voxels along short column segments times the 2-nonzeros-per-ray-and-column weight block is a real
// matrix product.  A ray's two taps in a column are in adjacent rows, so every group of four consecutive rows of a column
// holds at most two of them: exactly the 2:4 structure the sparse MMA skips, which runs 32 voxels per instruction at 9.7 clk
// against 16 voxels at 8.7 clk for the dense mma.sync (measured, profiles/r2_microbench.md).
//
// Block shape.  K = 32 voxels = 4 adjacent columns (of the stepping axis) x an 8-row window each; M = 16 rays = 4 adjacent
// bins of each of up to FOUR adjacent base angles (a "strip" of an angle group); N = 8 batch entries = half a 16-entry block of
// (slice, coefficient).  Four bins of one angle span at most 3*sqrt2 + 2 rows at a column, and the rays of the neighbouring
// angles that lie in the same strip of the detector stay within the 8-row window: 64 of the 512 weights are non-zero, 256 are
// stored.  Windows are clamped to the tile, so taps outside the tile (which belong to other tiles) simply have no row.
// When the angles of a group are too far apart for one window (coarse angular sampling), or the grouping leaves five bins of
// an angle in a strip, the item falls apart into pairs or single angles -- decided by the item builder, never a wrong result.
//
// Precision.  Operands are split bf16 pairs: F = Fh + Fl (tile, once per CTA), W = Wh + Wl (per weight), and
// D += Wh Fh + Wh Fl + Wl Fh with fp32 accumulation: relative error about 3 * 2^-18 = 1.1e-5 per product, inside the 1e-4
// per-operator tolerance.  cp4d_set_projector_mode selects the exact-fp32 gather instead.
//
// Work split.  CTA = (32 x 32 tile, pass, group of NB16 16-entry batch blocks); pass 0 = base angles whose rays step over
// columns, pass 1 = the others on the transposed tile, so one code path serves both.  The tile sits in shared memory as
// [block][hi/lo][8-entry half][column][33 rows] x 16 B, which makes every 8 x 8 ldmatrix operand 128 contiguous bytes.  The work
// items (angle group, strip, column range, window starts) are built once per context by k_fm_build; warps draw them from a
// shared counter; partial ray sums go to P[z][i][b][j] as 8-byte REDs.
#include <cuda_bf16.h>

#include <algorithm>
#include <cmath>

#include "cp4d_internal.cuh"
#include "device_helpers.cuh"

namespace cp4d {

namespace {

static_assert(TILE == 32, "the tile staging decodes indices with shifts for TILE = 32");
constexpr int FM_THREADS = 512;
constexpr int FM_STRIPS = WIN / 4 + 2;                 // strips -1 .. WIN/4 of four window bins
constexpr int FM_COL = (TILE + 1) * 16;                // bytes of one tile column: 32 rows x 16 B + 16 B of padding, so that the
                                                       // staging stores of one row across 8 columns hit 8 different bank groups
constexpr int FM_PLANE = 2 * TILE * FM_COL;            // bytes of one (block, hi/lo) plane: [half][column][row] x 16 B
constexpr float FM_KC = 0.5f * (TILE - 1);             // reference column where the two angles of a pair are aligned
constexpr float FM_SPAN = 5.99f;                       // largest spread of first-tap rows an 8-row window holds

struct FmArgs {
    int n, nz, nd, n0, m, mshift, gp, gpl;
    int tiles, agroups;
    int zper, z_base;          // slices per CTA = NB16 * 16 / m; first slice of this launch
    float margin;              // bins a ray of another angle of a group can sit from the first angle's bin of its touch point
    const TileGeo *geo;
    const FwAngle *fwang;
    const int4 *groups;        // [pass 0 groups | pass 1 groups]: up to four adjacent base angles, the one with the smallest |1/ss|
                               // first, -1 for an absent one
    int ngroups0, ngroups1;
    unsigned *items;           // work items of every (tile, pass), built once per context by k_fm_build: slot of (tile, pass) =
                               // 12 words x item_cap(pass) at word offset 12 (tile (cap0 + cap1) + (pass ? cap0 : 0)); long items
                               // from the front, short ones from the back
    int2 *counts;              // [tile][pass]: (long, short) items in the slot
    int cap0, cap1;            // item capacity of a slot = 4 FM_STRIPS groups of the pass
};

// per-CTA record of one angle group (shared memory): the per-angle tables and this tile's window geometry, plus what the
// strip bookkeeping needs, so that an item's setup is a handful of FMAs.  Absent angles repeat angle 0 with ia = -1.
struct FmGroup {
    float inv[4], step[4], delta[4];            // 1/ss, -cc/ss, window offset of the tile
    float istep[4];                             // 1/step (0 when the rays run along the columns)
    float r0[4], rinv[4];                       // bin ub of angle x sits, at the reference column, at angle-0 bin coordinate
                                                // ub / rinv[x] + r0[x]
    int ia[4], bstart[4];
};
constexpr int FM_MAXG = 128;                           // angle groups of a pass whose records a CTA keeps in shared memory (16 KB)
constexpr int FM_BUILDG = 32;                          // groups per round of the item builder
constexpr int FM_ITEMW = 12;                           // 32-bit words per work item
constexpr int FM_LONG = 14;                            // columns from which an item counts as long

// columns k in [0, TILE) where a ray group whose first-tap rows lie in [ylo + k st, yhi + k st] touches rows 0 .. TILE-1:
// ylo + k st < TILE and yhi + k st > -1
__device__ __forceinline__ void col_range(float ylo, float yhi, float st, float ist, int &klo, int &khi) {
    if (ist != 0.0f) {
        const float ka = ((float)TILE - ylo) * ist, kb = (-1.0f - yhi) * ist;     // st > 0: k < ka, k > kb; st < 0: reversed
        // integer k strictly inside (lo, hi); the 1e-3 keeps a column whose bound is an integer up to rounding
        klo = max(0, (int)floorf((st > 0.f ? kb : ka) + (1.0f - 1e-3f)));
        khi = min(TILE - 1, (int)ceilf((st > 0.f ? ka : kb) - (1.0f - 1e-3f)));
    } else if (ylo < (float)TILE && yhi > -1.0f) {
        klo = 0; khi = TILE - 1;
    } else {
        klo = TILE; khi = -1;
    }
}

// One work item of a (tile, pass), three words built once per context by k_fm_build (the geometry does not change):
//   w0 = (group in pass << 4 | strip + 1) | klo << 16 | khi << 24    columns of the tile the item's rays touch
//   w1 = bs1 | bs2 << 8 | bs3 << 16 (signed bytes) | used << 24       first window bin of angles 1-3 in this strip; angles in use
//   w2 = 4 | cnt1 << 4 | cnt2 << 8 | cnt3 << 12 | hb << 16            bins per angle; hb = four nibbles, one per half block of
//                                                                     four ray slots: angle | 4 (bins 4-7 of a long single) | 8 (valid)
//   w3 = 0;  w4 .. w11 = 16 x (qa | qb << 8)                          first row of the 8-row window at the two columns of step s
// Half blocks 0, 1 are the 8 rays of the first MMA column block, 2, 3 those of the second (only items of 3 or 4 angles).

// the shared-memory record of one angle group for one tile
__device__ __forceinline__ void fm_group_record(const FmArgs &a, const TileGeo *geo, const int4 gr, FmGroup &R, FwAngle &A0, TileGeo &G0) {
    const int idx[4] = {gr.x, gr.y, gr.z, gr.w};
    A0 = a.fwang[gr.x];
    G0 = geo[gr.x];
#pragma unroll
    for (int x = 0; x < 4; ++x) {
        const int i = idx[x] >= 0 ? idx[x] : gr.x;
        const FwAngle A = a.fwang[i];
        const TileGeo G = geo[i];
        R.inv[x] = A.inv; R.step[x] = A.step; R.delta[x] = G.delta;
        R.istep[x] = fabsf(A.step) > 1e-6f ? 1.0f / A.step : 0.0f;
        // ray ub of angle x sits, at the reference column, at angle-0 bin coordinate phi = ub inv_x / inv_0 + r0
        R.r0[x] = (FM_KC * (A.step - A0.step) - G.delta * A.inv) / A0.inv + G0.delta;
        R.rinv[x] = A0.inv / A.inv;
        R.ia[x] = idx[x]; R.bstart[x] = G.bstart;
    }
}

// Builds the work items of one (tile, pass) into its global slot (once per context: they depend on the geometry only).
__global__ void __launch_bounds__(FM_THREADS, 1) k_fm_build(FmArgs a) {
    __shared__ int s_nlong, s_nshort, s_ncand;
    __shared__ __align__(16) FmGroup s_grp[FM_BUILDG];
    __shared__ unsigned char s_t0[FM_BUILDG], s_tn[FM_BUILDG];      // first strip (+1) and number of strips of each group
    __shared__ unsigned short s_cand[FM_BUILDG * FM_STRIPS];        // candidate -> (group in round << 4) | (strip + 1)
    const int tile_id = blockIdx.x, pass = blockIdx.y, lane = threadIdx.x & 31;
    const TileGeo *geo = a.geo + (int64_t)tile_id * a.n0;
    const int pbeg = pass ? a.ngroups0 : 0, p1 = pbeg + (pass ? a.ngroups1 : a.ngroups0);
    const int cap = pass ? a.cap1 : a.cap0;
    unsigned *slot = a.items + FM_ITEMW * ((size_t)tile_id * (a.cap0 + a.cap1) + (pass ? a.cap0 : 0));
    if (threadIdx.x == 0) { s_nlong = 0; s_nshort = 0; }
    for (int pc = pbeg; pc < p1; pc += FM_BUILDG) {
        const int npc = min(FM_BUILDG, p1 - pc);
        __syncthreads();
        if ((int)threadIdx.x < npc) {
            FwAngle A0;
            TileGeo G0;
            fm_group_record(a, geo, a.groups[pc + threadIdx.x], s_grp[threadIdx.x], A0, G0);
            // strips that can hold a ray touching the tile: angle-0 window coordinates of the tile corners, widened by the
            // distance a ray of another angle can sit from the bin of its touch point at the reference column (a.margin)
            const float ss = 1.0f / A0.inv, cc = -A0.step * ss, e = (float)(TILE - 1);
            const float umin = G0.delta + fminf(0.f, e * cc) + fminf(0.f, e * ss), umax = G0.delta + fmaxf(0.f, e * cc) + fmaxf(0.f, e * ss);
            const int tf = max(-1, (int)floorf((umin - a.margin + 0.5f) * 0.25f)), tl = min(FM_STRIPS - 2, (int)floorf((umax + a.margin + 0.5f) * 0.25f));
            s_t0[threadIdx.x] = (unsigned char)(tf + 1);
            s_tn[threadIdx.x] = (unsigned char)max(0, tl - tf + 1);
        }
        __syncthreads();
        if (threadIdx.x < 32) {                              // candidate table: groups in order, their strips in order
            int base = 0;
            for (int q0 = 0; q0 < npc; q0 += 32) {
                const int q = q0 + lane, n = q < npc ? s_tn[q] : 0;
                int incl = n;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int v = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lane >= o) incl += v;
                }
                for (int r = 0; r < n; ++r) s_cand[base + incl - n + r] = (unsigned short)((q << 4) | (s_t0[q] + r));
                base += __shfl_sync(0xffffffffu, incl, 31);
            }
            if (lane == 0) s_ncand = base;
        }
        __syncthreads();
        // ---- work items: every candidate (group, strip) is examined by one thread: each angle's group of bins in the strip,
        // the columns its rays touch, and whether one 8-row window per column holds all angles (one item: 8 rays per MMA for two
        // angles, 16 for three or four), else the first two and the remaining angles are tried as pairs, else one item per angle ----
        for (int cnd = threadIdx.x; cnd < s_ncand; cnd += FM_THREADS) {
            const unsigned uu = s_cand[cnd];
            const FmGroup &R = s_grp[uu >> 4];
            const unsigned gg = (unsigned)(pc - pbeg) + (uu >> 4);          // group index within the pass
            const int ts = (int)(uu & 15) - 1;
            const float ft4 = 4.0f * (float)ts;
            int bs[4], cnt[4], ka[4], kb[4];
            float lo[4], hi[4], stp[4];
            unsigned ex = 0;                                   // angles with a ray that touches the tile in this strip
#pragma unroll
            for (int x = 0; x < 4; ++x) {
                bs[x] = 4 * ts; cnt[x] = 4;
                if (x > 0) {
                    // bin ub of angle x belongs to the strip whose extent [4 ts - 0.5, 4 ts + 3.5) holds phi(ub): the extents tile the
                    // line and both ends use the same expression, so every bin is in exactly one strip
                    const float r0 = R.r0[x], ri = R.rinv[x];
                    bs[x] = (int)ceilf((ft4 - 0.5f - r0) * ri);
                    cnt[x] = R.ia[x] >= 0 ? (int)ceilf((ft4 + 3.5f - r0) * ri) - bs[x] : 0;
                }
                // first-tap row of window bin ub of angle x at column k:  (ub - delta) inv + k step
                const float inv = R.inv[x], y0 = ((float)bs[x] - R.delta[x]) * inv, y1 = fmaf((float)(max(cnt[x], 1) - 1), inv, y0);
                lo[x] = fminf(y0, y1); hi[x] = fmaxf(y0, y1); stp[x] = R.step[x];
                ka[x] = TILE; kb[x] = -1;
                if (cnt[x] > 0 && bs[x] + cnt[x] > 0 && bs[x] < WIN) col_range(lo[x], hi[x], stp[x], R.istep[x], ka[x], kb[x]);
                if (ka[x] <= kb[x]) ex |= 1u << x;
                bs[x] = max(-100, min(100, bs[x])); cnt[x] = min(cnt[x], 8);
            }
            // columns of a set of angles and whether one window per column holds them: the spread of first-tap rows is convex
            // in k, so the two end columns decide
            auto cols = [&](unsigned S, int &fa, int &fb) {
                fa = TILE; fb = -1;
#pragma unroll
                for (int x = 0; x < 4; ++x)
                    if (S >> x & 1) { fa = min(fa, ka[x]); fb = max(fb, kb[x]); }
            };
            auto fits = [&](unsigned S) {
                int ia_, ib_;
                cols(S, ia_, ib_);
                const float fa = (float)ia_, fb = (float)ib_;
                float ha = -1e30f, la = 1e30f, hb_ = -1e30f, lb = 1e30f;
                bool ok = true;
#pragma unroll
                for (int x = 0; x < 4; ++x)
                    if (S >> x & 1) {
                        ok = ok && cnt[x] <= 4;
                        ha = fmaxf(ha, fmaf(fa, stp[x], hi[x])); la = fminf(la, fmaf(fa, stp[x], lo[x]));
                        hb_ = fmaxf(hb_, fmaf(fb, stp[x], hi[x])); lb = fminf(lb, fmaf(fb, stp[x], lo[x]));
                    }
                return ok && ha - la < FM_SPAN && hb_ - lb < FM_SPAN;
            };
            // long items are handed out first (front of the list), short ones last (stored from the back): an even finish
            auto push = [&](unsigned S, unsigned hb) {
                int fa, fb;
                cols(S, fa, fb);
                const bool lng = fb - fa >= FM_LONG;
                const int at = lng ? atomicAdd(&s_nlong, 1) : cap - 1 - atomicAdd(&s_nshort, 1);
                unsigned *it = slot + FM_ITEMW * (size_t)at;
                it[0] = (gg << 4) | (uu & 15u) | ((unsigned)fa << 16) | ((unsigned)fb << 24);
                it[1] = ((unsigned)bs[1] & 0xffu) | (((unsigned)bs[2] & 0xffu) << 8) | (((unsigned)bs[3] & 0xffu) << 16) | (S << 24);
                it[2] = 4u | ((unsigned)cnt[1] << 4) | ((unsigned)cnt[2] << 8) | ((unsigned)cnt[3] << 12) | (hb << 16);
                it[3] = 0u;
                // window start of every step (four columns from fa & ~3 on): floor of the lowest first-tap row of the item's angles
                // at each column, clamped into the tile
                auto wstart = [&](float fk) {
                    float l = 1e6f;
#pragma unroll
                    for (int x = 0; x < 4; ++x)
                        if (S >> x & 1) l = fminf(l, fmaf(fk, stp[x], lo[x]));
                    return (unsigned)min(max((int)floorf(l), 0), TILE - 8);
                };
                for (int w = 0; w < 8; ++w) {
                    const float fk = (float)((fa & ~3) + 4 * w);
                    it[4 + w] = wstart(fk) | (wstart(fk + 1.0f) << 8) | (wstart(fk + 2.0f) << 16) | (wstart(fk + 3.0f) << 24);
                }
            };
            auto nibbles = [&](unsigned S) {                   // the angles of S on consecutive half blocks
                unsigned hb = 0;
                int h = 0;
#pragma unroll
                for (int x = 0; x < 4; ++x)
                    if (S >> x & 1) { hb |= (8u | (unsigned)x) << (4 * h); ++h; }
                return hb;
            };
            auto singles = [&](unsigned S) {
#pragma unroll
                for (int x = 0; x < 4; ++x)
                    if (S >> x & 1) push(1u << x, (8u | (unsigned)x) | (cnt[x] > 4 ? (12u | (unsigned)x) << 4 : 0u));
            };
            auto pair_or_singles = [&](unsigned S) {
                if (__popc(S) == 2 && fits(S)) push(S, nibbles(S));
                else singles(S);
            };
            const int nex = __popc(ex);
            if (nex >= 2 && fits(ex)) {
                push(ex, nibbles(ex));
            } else if (nex >= 3) {
                const unsigned first = ex & (0u - ex), rest = ex ^ first, second = rest & (0u - rest);
                pair_or_singles(first | second);
                pair_or_singles(ex ^ (first | second));
            } else {
                singles(ex);
            }
        }
        __syncthreads();
    }
    __syncthreads();
    if (threadIdx.x == 0) a.counts[tile_id * 2 + pass] = make_int2(s_nlong, s_nshort);
}

template <int NB16>
__global__ void __launch_bounds__(FM_THREADS, 1) k_forward_mma(const float *__restrict__ f, float *__restrict__ P, FmArgs a) {
    extern __shared__ __align__(128) unsigned char tile[];     // [NB16][2][2][TILE][TILE + 1] x 16 B
    __shared__ int s_next;
    __shared__ __align__(16) FmGroup s_grp[FM_MAXG];
    const int tiles_1d = (a.n + TILE - 1) / TILE;
    const int tile_id = blockIdx.x % a.tiles, ag = blockIdx.x / a.tiles;
    const int pass = blockIdx.y & 1, z0 = a.z_base + (blockIdx.y >> 1) * a.zper;
    const int x0 = (tile_id % tiles_1d) * TILE, y0 = (tile_id / tiles_1d) * TILE;

    // ---- stage the tile: fp32 -> (hi, lo) bf16, pass coordinates (column = stepping axis); 4 entries (8 loads) in flight ----
    constexpr int N_ENT = NB16 * 2 * TILE * TILE;
    static_assert(N_ENT % (4 * FM_THREADS) == 0, "staging loop is unrolled by 4");
    for (int e0 = threadIdx.x; e0 < N_ENT; e0 += 4 * FM_THREADS) {
        float4 q[4][2];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int e = e0 + r * FM_THREADS;
            // pass 1: 32 consecutive threads take the 32 rows (= x) of one column; pass 0: 16 consecutive columns (= x) of one
            // row for each half -- either way a warp reads 1 KB of contiguous global memory per load pair
            const int zb = e >> 11;
            const int row = pass ? e & (TILE - 1) : (e >> 6) & (TILE - 1);
            const int kcol = pass ? (e >> 5) & (TILE - 1) : (e & 15) | ((e >> 1) & 16);
            const int jh = pass ? (e >> 10) & 1 : (e >> 4) & 1;
            const int gx = x0 + (pass ? row : kcol), gy = y0 + (pass ? kcol : row);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int flat = zb * 16 + jh * 8 + h * 4, sl = z0 + (flat >> a.mshift), j = flat & (a.m - 1);
                q[r][h] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (gx < a.n && gy < a.n && sl < a.nz)
                    q[r][h] = __ldg(reinterpret_cast<const float4 *>(f + (((int64_t)sl * a.n + gy) * a.n + gx) * a.m + j));
            }
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int e = e0 + r * FM_THREADS;
            // pass 1: 32 consecutive threads take the 32 rows (= x) of one column; pass 0: 16 consecutive columns (= x) of one
            // row for each half -- either way a warp reads 1 KB of contiguous global memory per load pair
            const int zb = e >> 11;
            const int row = pass ? e & (TILE - 1) : (e >> 6) & (TILE - 1);
            const int kcol = pass ? (e >> 5) & (TILE - 1) : (e & 15) | ((e >> 1) & 16);
            const int jh = pass ? (e >> 10) & 1 : (e >> 4) & 1;
            uint4 hi, lo;
            split2(q[r][0].x, q[r][0].y, hi.x, lo.x); split2(q[r][0].z, q[r][0].w, hi.y, lo.y);
            split2(q[r][1].x, q[r][1].y, hi.z, lo.z); split2(q[r][1].z, q[r][1].w, hi.w, lo.w);
            unsigned char *dst = tile + (size_t)(zb * 2) * FM_PLANE + (jh * TILE + kcol) * FM_COL + row * 16;
            *reinterpret_cast<uint4 *>(dst) = hi;
            *reinterpret_cast<uint4 *>(dst + FM_PLANE) = lo;
        }
    }

    const int pbeg = pass ? a.ngroups0 : 0, pcnt = pass ? a.ngroups1 : a.ngroups0;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const unsigned tile_s = (unsigned)__cvta_generic_to_shared(tile);
    // ldmatrix row address of this lane: matrix = lane / 8 = column of the step, row lane & 7 of its window
    const unsigned ld_base = tile_s + (lane >> 3) * FM_COL + ((lane & 7) << 4);
    const TileGeo *geo = a.geo + (int64_t)tile_id * a.n0;
    // epilogue: I add batch entries 8 half + 2 t, + 1 of block zb = coefficients j, j + 1 of slice sl; element offset of (sl, j) in P
    unsigned zoff[NB16][2];
    bool zok[NB16][2];
#pragma unroll
    for (int zb = 0; zb < NB16; ++zb)
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
            const int flat = zb * 16 + hf * 8 + 2 * t, sl = z0 + (flat >> a.mshift), j = flat & (a.m - 1);
            zok[zb][hf] = sl < a.nz;
            zoff[zb][hf] = (unsigned)sl * (unsigned)(a.n0 * a.gp) * (unsigned)a.m + (unsigned)j;
        }

    // ---- the records of all angle groups of this pass for this tile; the item list of (tile, pass) ----
    if (threadIdx.x == 0) s_next = 0;
    for (int q = threadIdx.x; q < pcnt; q += FM_THREADS) {
        FwAngle A0;
        TileGeo G0;
        fm_group_record(a, geo, a.groups[pbeg + q], s_grp[q], A0, G0);
    }
    __syncthreads();                                         // the tile is staged, the records are written
    {
        const int2 cnt = a.counts[tile_id * 2 + pass];
        const int n_long = cnt.x, n_items = cnt.x + cnt.y, cap = pass ? a.cap1 : a.cap0;
        const unsigned *slot = a.items + FM_ITEMW * ((size_t)tile_id * (a.cap0 + a.cap1) + (pass ? a.cap0 : 0));
        // warps draw items from one counter; small problems split the list over the agroups CTAs of a tile (item u of CTA ag
        // is list entry u agroups + ag, which keeps long and short items on every CTA).  The next item is fetched while the
        // current one runs
        auto fetch = [&](int &u, uint4 &w, unsigned &q) {      // q: lane s (< 8) gets the window starts of step s (4 columns)
            int v = 0;
            if (lane == 0) v = atomicAdd(&s_next, 1);
            u = __shfl_sync(0xffffffffu, v, 0) * a.agroups + ag;
            w = make_uint4(0u, 0u, 0u, 0u);
            q = 0u;
            if (u < n_items) {
                const unsigned *it = slot + FM_ITEMW * (size_t)(u < n_long ? u : cap - 1 - (u - n_long));
                w = __ldg(reinterpret_cast<const uint4 *>(it));
                q = __ldg(it + 4 + (lane & 7));
            }
        };
        int u, un;
        uint4 wi, wn;
        unsigned qi, qn;
        fetch(u, wi, qi);
        for (; u < n_items; u = un, wi = wn, qi = qn) {
            fetch(un, wn, qn);
            const unsigned w0 = wi.x, w1 = wi.y, w2 = wi.z;
            const FmGroup &R = s_grp[(w0 & 0xffffu) >> 4];
            const int ts = (int)(w0 & 15u) - 1, klo = (int)((w0 >> 16) & 0xffu), khi = (int)(w0 >> 24);
            const unsigned bspack = (w1 << 8) | ((unsigned)(4 * ts) & 0xffu);      // first bin of angle x: signed byte x
            const unsigned hb = w2 >> 16;
            // window start per column (the same for every lane): lane s holds the four bytes of step s (columns kb + 4 s .. + 3)
            // from the item; the loop fetches them with one shuffle
            const int kb = klo & ~3;
            const int nstep = ((khi - kb) >> 2) + 1;
            // The weight block is the sparse operand: A[16 rays x 32 voxels], voxel k = 8 c + r = row r of the 8-row window of
            // column c of the step; a ray has its two taps in adjacent rows, so every group of four rows holds at most two of
            // them (2:4).  Lane (g, t) computes, for rays g (slot g, "nb 0") and g + 8 ("nb 1"), the two kept elements of group t
            // (column t / 2, rows 4 (t & 1) .. + 3) and of group t + 4 (column 2 + t / 2, same rows).  Half block 2 nb + g / 4 of
            // the item names a ray's angle; its slots hold consecutive bins.
            int r_bub[2], r_x[2];
            bool r_ok[2];
            float r_step[2], r_y[2];       // first-tap row at column kb + t / 2, relative to the first row of my row half
#pragma unroll
            for (int nb = 0; nb < 2; ++nb) {
                const unsigned d = (hb >> (4 * (2 * nb + (g >> 2)))) & 15u;
                const int x = (int)(d & 3u), off = (int)(d & 4u) + (g & 3);
                const int bsx = (int)(bspack << (24 - 8 * x)) >> 24, cx = (int)((w2 >> (4 * x)) & 15u);
                r_x[nb] = x;
                r_bub[nb] = bsx + off;
                r_ok[nb] = (d & 8u) && off < cx && r_bub[nb] >= 0 && r_bub[nb] < WIN;
                r_step[nb] = R.step[x];
                r_y[nb] = r_ok[nb] ? fmaf((float)(kb + (t >> 1)), r_step[nb], ((float)r_bub[nb] - R.delta[x]) * R.inv[x]) - (float)(4 * (t & 1)) : -1e6f;
            }
            // ---- partial ray sums of this tile -> P[z][i][b][j]: element offsets of my two rays (see the epilogue) ----
            unsigned r_off[2];
#pragma unroll
            for (int nb = 0; nb < 2; ++nb) {
                const int b = R.bstart[r_x[nb]] + r_bub[nb];
                r_ok[nb] = r_ok[nb] && b >= 0 && b < a.nd;
                r_off[nb] = (unsigned)((R.ia[r_x[nb]] * a.gp + a.gpl + b) * a.m);
            }

            float acc[NB16][2][4];         // [batch block][8-entry half]: rays g (0, 1) and g + 8 (2, 3) x batch entries 2t, 2t + 1
#pragma unroll
            for (int zb = 0; zb < NB16; ++zb)
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) acc[zb][hf][0] = acc[zb][hf][1] = acc[zb][hf][2] = acc[zb][hf][3] = 0.f;

            const unsigned qsel = 0x4440u + (unsigned)(t >> 1), qsel2 = qsel + 2u;       // byte t / 2 (resp. 2 + t / 2) of the step's word
            const unsigned msel = 0x4440u + (lane >> 3);                                  // byte of my ldmatrix column
            unsigned adr_k = ld_base + (unsigned)kb * FM_COL;
            float ys[2][2] = {{r_y[0], fmaf(2.0f, r_step[0], r_y[0])}, {r_y[1], fmaf(2.0f, r_step[1], r_y[1])}};   // [nb][column]
            const float st4[2] = {4.0f * r_step[0], 4.0f * r_step[1]};
            for (int st = 0; st < nstep; ++st, adr_k += 4 * FM_COL) {
                const unsigned qw = __shfl_sync(0xffffffffu, qi, st);
                const float fq[2] = {(float)__byte_perm(qw, 0u, qsel), (float)__byte_perm(qw, 0u, qsel2)};
                unsigned ah[4], al[4];
                float nib[4];
#pragma unroll
                for (int cc = 0; cc < 2; ++cc)
#pragma unroll
                    for (int nb = 0; nb < 2; ++nb) {
                        // row of the first tap relative to my row half; the kept pair starts at row i0 = clamp(floor(z), 0, 2)
                        const float z = ys[nb][cc] - fq[cc];
                        const float i0 = fminf(fmaxf(floorf(z), 0.0f), 2.0f);
                        const float dd = z - i0;
                        nib[2 * cc + nb] = fmaf(5.0f, i0, 4.0f);                          // positions (i0, i0 + 1), two bits each: 4, 9, 14
                        split2(__saturatef(1.0f - fabsf(dd)), __saturatef(1.0f - fabsf(dd - 1.0f)), ah[2 * cc + nb], al[2 * cc + nb]);
                        ys[nb][cc] += st4[nb];
                    }
                // metadata: lane 4g wants the groups 0-3 (low half: ray g, high half: ray g + 8), lane 4g + 1 the groups 4-7
                // (a butterfly over the quad: first the lanes two apart, then lanes 0 and 1 hand each other what the other needs)
                unsigned e0 = (unsigned)__float2int_rn(fmaf(nib[1], 65536.0f, nib[0])) << (4 * t), e1 = (unsigned)__float2int_rn(fmaf(nib[3], 65536.0f, nib[2])) << (4 * t);
                e0 |= __shfl_xor_sync(0xffffffffu, e0, 2);
                e1 |= __shfl_xor_sync(0xffffffffu, e1, 2);
                const unsigned e = ((t & 1) ? e1 : e0) | __shfl_xor_sync(0xffffffffu, (t & 1) ? e0 : e1, 1);
                const unsigned adr = adr_k + (__byte_perm(qw, 0u, msel) << 4);
#pragma unroll
                for (int zb = 0; zb < NB16; ++zb)
#pragma unroll
                    for (int hf = 0; hf < 2; ++hf) {
                        unsigned bh[4], bl[4];
                        ldsm4t(bh, adr + zb * 2 * FM_PLANE + hf * (TILE * FM_COL));
                        ldsm4t(bl, adr + zb * 2 * FM_PLANE + FM_PLANE + hf * (TILE * FM_COL));
                        mma_sp16832(acc[zb][hf], ah, bh, e);
                        mma_sp16832(acc[zb][hf], ah, bl, e);
                        mma_sp16832(acc[zb][hf], al, bh, e);
                    }
            }
            // epilogue: my D entries are two consecutive batch entries of ray g and two of ray g + 8: one 8-byte RED each.  (One
            // 16-byte RED per lane after an exchange between lanes t and t ^ 1 halves the REDs, but its selects and shuffles cost
            // more than the REDs, which the kernel hides: 3.06 -> 3.01 ms.)
#pragma unroll
            for (int zb = 0; zb < NB16; ++zb)
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    const float (&d)[4] = acc[zb][hf];
                    if (r_ok[0] && zok[zb][hf]) atomicAdd(reinterpret_cast<float2 *>(P + (size_t)zoff[zb][hf] + r_off[0]), make_float2(d[0], d[1]));
                    if (r_ok[1] && zok[zb][hf]) atomicAdd(reinterpret_cast<float2 *>(P + (size_t)zoff[zb][hf] + r_off[1]), make_float2(d[2], d[3]));
                }
        }
    }
}

// slices [z_base, z_base + nz_part) in groups of NB16 batch blocks per CTA
template <int NB16>
cudaError_t fm_launch(cp4d_ctx *c, const float *f, float *P, FmArgs a, int z_base, int nz_part) {
    const Dims &d = c->d;
    a.zper = NB16 * 16 / d.m;
    a.z_base = z_base;
    const int zgroups = (nz_part + a.zper - 1) / a.zper;
    // small problems: split the item list of a (tile, pass) over up to 8 CTAs so that every SM has work
    const int64_t ctas = (int64_t)d.tiles * 2 * zgroups;
    a.agroups = (int)std::max<int64_t>(1, std::min<int64_t>(8, 148 / ctas));
    const dim3 grid(d.tiles * a.agroups, 2 * zgroups);
    k_forward_mma<NB16><<<grid, FM_THREADS, (size_t)NB16 * 2 * FM_PLANE, c->stream>>>(f, P, a);
    return cudaGetLastError();
}

}  // namespace

bool forward_mma_supported(const Dims &d) {
    if ((int64_t)d.nz * d.n0 * d.nd * d.m >= (int64_t)1 << 31) return false;      // the epilogue keeps 32-bit element offsets into P
    return (d.m == 4 || d.m == 8 || d.m == 16 || d.m == 32);
}

// CP4D_PROJ_AUTO: the tensor kernel runs one 512-thread CTA per SM and pays a tile staging and a work-item build per CTA, so it
// only wins once (tile, pass, batch group) CTAs fill the GPU; below that the fp32 gather is faster (config 2: 85 vs 74 us)
bool forward_mma_preferred(const Dims &d) {
    if (!forward_mma_supported(d)) return false;
    const int blocks_total = (d.nz * d.m + 15) / 16, nb = d.m == 32 ? 2 : std::min(3, blocks_total);
    const int64_t ctas = (int64_t)d.tiles * 2 * ((blocks_total + nb - 1) / nb);
    return ctas >= 148;
}

cudaError_t forward_mma_init() {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(k_forward_mma<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 1 * 2 * FM_PLANE)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_forward_mma<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 2 * FM_PLANE)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_forward_mma<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, 3 * 2 * FM_PLANE);
}

// largest group of adjacent base angles whose rays one strip bookkeeping serves: a ray of another angle that touches the tile
// sits, at the tile's middle column, at most (gs - 1) 16 sqrt2 sin(pi/n0) bins outside the first angle's window, which the two
// spare strips (bins -4 .. -1 and 48 .. 51) absorb for n0 >= 24 (pairs) and n0 >= 72 (four).  Coarser sets: every angle on its own.
static int fm_group_size(int n0) { return n0 >= 72 ? 4 : n0 >= 24 ? 2 : 1; }

// host: group adjacent base angles of one pass (same stepping axis, same sign of 1/ss, consecutive indices); the angle with
// the smallest |1/ss| comes first, so that a strip of four of its bins holds at most four bins of each of the others
int forward_mma_groups(const FwAngle *fw, const int32_t *order, int n0, int n_colstep, int4 *out, int *ngroups0, int *ngroups1) {
    int n = 0;
    const int gs = fm_group_size(n0);
    for (int pass = 0; pass < 2; ++pass) {
        const int l0 = pass ? n_colstep : 0, l1 = pass ? n0 : n_colstep;
        const int start = n;
        for (int q = l0; q < l1;) {
            int idx[4] = {order[q], -1, -1, -1}, cnt = 1;
            while (cnt < gs && q + cnt < l1 && order[q + cnt] == order[q] + cnt && (fw[order[q]].inv > 0.f) == (fw[order[q + cnt]].inv > 0.f)) {
                idx[cnt] = order[q + cnt];
                ++cnt;
            }
            std::stable_sort(idx, idx + cnt, [&](int x, int y) { return std::fabs(fw[x].inv) < std::fabs(fw[y].inv); });
            out[n++] = make_int4(idx[0], idx[1], idx[2], idx[3]);
            q += cnt;
        }
        *(pass ? ngroups1 : ngroups0) = n - start;
    }
    return n;
}

static FmArgs fm_args(const cp4d_ctx *c) {
    const Dims &d = c->d;
    int ms = 0;
    while ((1 << ms) < d.m) ++ms;
    // 1.5 bins for the taps and the half-bin extents + (TILE/2) sqrt2 sin(pi/n0) per angle step for the drift over half a tile
    const float margin = 1.5f + (float)(fm_group_size(d.n0) - 1) * 0.5f * TILE * 1.41421356f * std::sin(3.14159265f / (float)d.n0);
    return FmArgs{d.n, d.nz, d.nd, d.n0, d.m, ms, d.nd, 0, d.tiles, 1, 0, 0, margin, c->geo, c->fwang, c->fw_groups, c->n_groups0, c->n_groups1,
                  c->fw_items, c->fw_counts, 4 * FM_STRIPS * c->n_groups0, 4 * FM_STRIPS * c->n_groups1};
}

// item slots of a context: every (group, strip) of a tile may fall apart into four single-angle items; the groups of both
// passes together are at most n0 / group size + 8 (a pass ends, the sign of 1/ss changes or the order jumps at most 8 times)
uint64_t forward_mma_item_bytes(const Dims &d) {
    if (!forward_mma_supported(d)) return 0;
    return (uint64_t)d.tiles * 4 * FM_STRIPS * (uint64_t)(d.n0 / fm_group_size(d.n0) + 8) * (FM_ITEMW * 4);
}

// the tensor kernel can run in this context: supported shape, the group records of a pass fit its shared memory, and the
// groups fit the item slots (cp4d_create: after forward_mma_groups)
bool forward_mma_usable(const cp4d_ctx *c) {
    return forward_mma_supported(c->d) && c->fw_items != nullptr && c->n_groups0 <= FM_MAXG && c->n_groups1 <= FM_MAXG &&
           c->n_groups0 + c->n_groups1 <= c->d.n0 / fm_group_size(c->d.n0) + 8;
}

// cp4d_create: the work items of every (tile, pass), once (they depend on the geometry only)
cudaError_t forward_mma_build(cp4d_ctx *c) {
    if (!forward_mma_usable(c)) return cudaSuccess;
    k_fm_build<<<dim3(c->d.tiles, 2), FM_THREADS, 0, c->stream>>>(fm_args(c));
    return cudaGetLastError();
}

cudaError_t launch_forward_mma(cp4d_ctx *c, const float *f, float *P) {
    const Dims &d = c->d;
    const FmArgs a = fm_args(c);
    // 16-entry batch blocks per CTA: three (192 KB of shared memory) unless the volume has fewer; m = 32 needs whole slices.
    // Slices that do not fill a last group of three blocks go to a second launch with one or two blocks per CTA (config 3:
    // 32 slices = 10 x 3 + 2), instead of a group that multiplies a block of zeros
    const int blocks_total = (d.nz * d.m + 15) / 16;
    if (d.m == 32) return fm_launch<2>(c, f, P, a, 0, d.nz);
    const int spb = 16 / d.m;                                   // slices per block
    const int full = blocks_total / 3, rem = blocks_total % 3;
    cudaError_t e = cudaSuccess;
    if (full > 0) e = fm_launch<3>(c, f, P, a, 0, std::min(d.nz, full * 3 * spb));
    if (e != cudaSuccess || rem == 0) return e;
    if (full > 0) c->launches++;
    const int zb = full * 3 * spb;
    return rem == 1 ? fm_launch<1>(c, f, P, a, zb, d.nz - zb) : fm_launch<2>(c, f, P, a, zb, d.nz - zb);
}

}  // namespace cp4d
