// Forward projector on the tensor cores (Eq. 9, with the pi-fold of L198-L202): the Joseph ray sums of all
// coefficients over the base angles, as small dense products  D[16 batch entries x 8 rays] += F[16 x 16 voxels] * W[16 voxels x 8 rays].
//
// Why.  The CUDA-core gather (projectors.cu) needs one shared-memory word per FMA and sits on the LSU data pipe at 0.19 of
// the FP32 peak.  The interpolation weights do not depend on the slice or on the coefficient, so the batch axis (slice, j) is
// a dense axis: a block of 16 voxels along a short column segment times the 2-nonzeros-per-ray weight block is a real matrix
// product.  mma.sync (HMMA.16816) measured 950 MAC/clk/SM on B200, 7.4x the FP32 FMA rate, and it does not touch the LSU pipe
// beyond one ldmatrix per 16 x 16 operand -- so a weight block that is 1/4 dense still wins.
//
// Block shape.  K = 16 voxels = 2 adjacent columns (of the stepping axis) x 8 consecutive rows; N = 8 rays = 4 adjacent bins of
// each of TWO adjacent base angles (a "strip pair"); M = 16 batch entries = (slices x coefficients) of one voxel.  Four bins of
// one angle span at most 3*sqrt2 + 2 rows at a column, and the rays of the neighbouring angle that lie in the same strip of the
// detector stay within one more row of them, so an 8-row window per column holds every tap: 32 of the 128 weights are
// non-zero.  Windows are clamped to the tile, so taps outside the tile (which belong to other tiles) simply have no row.
// When the two angles are too far apart for one window (coarse angular sampling), or the pairing leaves five bins of the
// second angle in a strip, the unit is processed as two single-angle units -- a warp-uniform decision, never a wrong result.
//
// Precision.  Operands are split bf16 pairs: F = Fh + Fl (tile, once per CTA), W = Wh + Wl (per weight), and
// D += Fh Wh + Fl Wh + Fh Wl with fp32 accumulation: relative error about 3 * 2^-18 = 1.1e-5 per product, inside the 1e-4
// per-operator tolerance.  cp4d_set_forward_mode selects the exact-fp32 gather instead.
//
// Work split.  CTA = (32 x 32 tile, pass, group of NB16 16-entry batch blocks); pass 0 = base angles whose rays step over
// columns, pass 1 = the others on the transposed tile, so one code path serves both.  The tile sits in shared memory as
// [block][hi/lo][8-entry half][column][row] x 16 B, which makes every 8 x 8 ldmatrix operand 128 contiguous bytes.  Warps
// draw units (angle pair, strip) from a shared counter; partial ray sums go to P[z][i][b][j] with scalar REDs (32-byte
// runs of 8 coefficients per bin).
#include <cuda_bf16.h>

#include <algorithm>
#include <cmath>

#include "cp4d_internal.cuh"
#include "device_helpers.cuh"

namespace cp4d {

namespace {

static_assert(TILE == 32, "the tile staging decodes indices with shifts for TILE = 32");
constexpr int FM_THREADS = 512;
constexpr int FM_WARPS = FM_THREADS / 32;
constexpr int FM_STRIPS = WIN / 4 + 2;                 // strips -1 .. WIN/4 of four window bins
constexpr int FM_PLANE = 2 * TILE * TILE * 16;         // bytes of one (block, hi/lo) plane: [half][column][row] x 16 B
constexpr float FM_KC = 0.5f * (TILE - 1);             // reference column where the two angles of a pair are aligned
constexpr float FM_SPAN = 5.99f;                       // largest spread of first-tap rows an 8-row window holds
constexpr int FM_STG = 20;                             // floats per ray of a warp's 8 x 16 epilogue patch (20: conflict-free stores)

struct FmArgs {
    int n, nz, nd, n0, m, mshift, gp, gpl;
    int tiles, agroups;
    int zper;                  // slices per CTA = NB16 * 16 / m
    float margin;              // bins a ray of the second angle of a pair can sit from the first angle's bin of its touch point
    const TileGeo *geo;
    const FwAngle *fwang;
    const int2 *pairs;         // [pass 0 pairs | pass 1 pairs]: (ia, ib), |inv(ib)| >= |inv(ia)|, ib = -1 for a single angle
    int npairs0, npairs1;
};

// per-CTA record of one angle pair (shared memory): the per-angle tables and this tile's window geometry, plus what the
// strip bookkeeping needs, so that a unit's setup is a handful of FMAs
struct FmPair {
    float inv0, step0, delta0, inva0;     // angle 0 (the one with the smaller |1/ss|): 1/ss, -cc/ss, window offset, 1/a
    float inv1, step1, delta1, inva1;     // angle 1 (= angle 0 for a single)
    float r0, rinv1, istep0, istep1;      // angle-1 bin ub1 sits at angle-0 bin coordinate (ub1 - s0) / rinv1, s0 = -r0 rinv1, at the
                                          // reference column; istep = 1/step (0 when the rays run along the columns)
    int ia, ib, bstart0, bstart1;
};
constexpr int FM_MAXP = 64;
constexpr int FM_MAXITEMS = 2 * FM_MAXP * FM_STRIPS;   // every (pair, strip) may fall apart into two items
constexpr int FM_LONG = 14;                           // columns from which an item counts as long               // pairs per chunk of a CTA's pair list

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

// one work item of a CTA: (angle pair, strip, which of the two angles) with its trimmed column range, built once per CTA by
// all threads in parallel so that a warp's per-item setup is a decode and a few FMAs
struct FmItem {
    unsigned short pair_strip;     // (pair << 4) | (strip + 1)
    unsigned char klo, khi;        // columns of the tile the strip's rays touch
    signed char b1s;               // first window bin of the second angle's group in this strip
    unsigned char cnt1;            // bins of that group
    unsigned char mode;            // 0: both angles in one window (slots 0-3 / 4-7), 1: first angle only, 2: second angle only
    unsigned char pad;
};
static_assert(sizeof(FmItem) == 8, "FmItem is one 8-byte shared-memory word");

template <int NB16>
__global__ void __launch_bounds__(FM_THREADS, 1) k_forward_mma(const float *__restrict__ f, float *__restrict__ P, FmArgs a) {
    extern __shared__ __align__(128) unsigned char tile[];     // [NB16][2][2][TILE][TILE] x 16 B
    __shared__ int s_next, s_nlong, s_nshort, s_ncand;
    __shared__ __align__(16) float s_stg[FM_WARPS][8 * FM_STG];
    __shared__ __align__(16) FmPair s_pair[FM_MAXP];
    __shared__ unsigned char s_t0[FM_MAXP], s_tn[FM_MAXP];      // first strip (+1) and number of strips of each pair
    __shared__ unsigned short s_cand[FM_MAXP * FM_STRIPS];      // candidate -> (pair << 4) | (strip + 1)
    __shared__ __align__(8) FmItem s_item[FM_MAXITEMS];
    float *stg = s_stg[threadIdx.x >> 5];
    const int tiles_1d = (a.n + TILE - 1) / TILE;
    const int tile_id = blockIdx.x % a.tiles, ag = blockIdx.x / a.tiles;
    const int pass = blockIdx.y & 1, z0 = (blockIdx.y >> 1) * a.zper;
    const int x0 = (tile_id % tiles_1d) * TILE, y0 = (tile_id / tiles_1d) * TILE;

    // ---- stage the tile: fp32 -> (hi, lo) bf16, pass coordinates (column = stepping axis); 4 entries (8 loads) in flight ----
    constexpr int N_ENT = NB16 * 2 * TILE * TILE;
    static_assert(N_ENT % (4 * FM_THREADS) == 0, "staging loop is unrolled by 4");
    for (int e0 = threadIdx.x; e0 < N_ENT; e0 += 4 * FM_THREADS) {
        float4 q[4][2];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int e = e0 + r * FM_THREADS;
            const int row = e & (TILE - 1), kcol = (e >> 5) & (TILE - 1), jh = (e >> 10) & 1, zb = e >> 11;
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
            const int row = e & (TILE - 1), kcol = (e >> 5) & (TILE - 1), jh = (e >> 10) & 1, zb = e >> 11;
            uint4 hi, lo;
            split2(q[r][0].x, q[r][0].y, hi.x, lo.x); split2(q[r][0].z, q[r][0].w, hi.y, lo.y);
            split2(q[r][1].x, q[r][1].y, hi.z, lo.z); split2(q[r][1].z, q[r][1].w, hi.w, lo.w);
            unsigned char *dst = tile + (size_t)(zb * 2) * FM_PLANE + ((jh * TILE + kcol) * TILE + row) * 16;
            *reinterpret_cast<uint4 *>(dst) = hi;
            *reinterpret_cast<uint4 *>(dst + FM_PLANE) = lo;
        }
    }

    // ---- this CTA's share of the pass's angle pairs, in chunks of FM_MAXP ----
    const int pbeg = pass ? a.npairs0 : 0, pcnt = pass ? a.npairs1 : a.npairs0;
    const int p0 = pbeg + (int)((int64_t)pcnt * ag / a.agroups), p1 = pbeg + (int)((int64_t)pcnt * (ag + 1) / a.agroups);
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const unsigned tile_s = (unsigned)__cvta_generic_to_shared(tile);
    // ldmatrix row address of this lane: matrix = lane / 8 -> (column k0 + matrix / 2, half matrix & 1), row lane & 7
    const unsigned ld_half = (lane >> 3) & 1, ld_col = lane >> 4, ld_row = lane & 7;
    const unsigned ld_base = tile_s + (((ld_half * TILE + ld_col) * TILE + ld_row) << 4);
    const TileGeo *geo = a.geo + (int64_t)tile_id * a.n0;

    const int n_chunk = (p1 - p0 + FM_MAXP - 1) / FM_MAXP, per_chunk = n_chunk ? (p1 - p0 + n_chunk - 1) / n_chunk : 0;   // even chunks
    for (int pc = p0; pc < p1; pc += per_chunk) {
        const int npc = min(per_chunk, p1 - pc);
        __syncthreads();                                     // the tile is staged / every warp is done with the previous chunk
        if ((int)threadIdx.x < npc) {
            const int2 pr = a.pairs[pc + threadIdx.x];
            const FwAngle A0 = a.fwang[pr.x], A1 = a.fwang[pr.y >= 0 ? pr.y : pr.x];
            const TileGeo G0 = geo[pr.x], G1 = geo[pr.y >= 0 ? pr.y : pr.x];
            FmPair R;
            R.inv0 = A0.inv; R.step0 = A0.step; R.delta0 = G0.delta; R.inva0 = A0.inv_a;
            R.inv1 = A1.inv; R.step1 = A1.step; R.delta1 = G1.delta; R.inva1 = A1.inv_a;
            // angle-1 ray ub1 sits, at the reference column, at angle-0 bin coordinate phi = r1 ub1 + r0
            const float r1 = A1.inv / A0.inv;
            R.r0 = (FM_KC * (A1.step - A0.step) - G1.delta * A1.inv) / A0.inv + G0.delta;
            R.rinv1 = 1.0f / r1;
            R.istep0 = fabsf(A0.step) > 1e-6f ? 1.0f / A0.step : 0.0f;
            R.istep1 = fabsf(A1.step) > 1e-6f ? 1.0f / A1.step : 0.0f;
            R.ia = pr.x; R.ib = pr.y; R.bstart0 = G0.bstart; R.bstart1 = G1.bstart;
            s_pair[threadIdx.x] = R;
            // strips that can hold a ray touching the tile: angle-0 window coordinates of the tile corners, widened by the
            // distance an angle-1 ray can sit from the bin of its touch point at the reference column (a.margin)
            const float ss = 1.0f / A0.inv, cc = -A0.step * ss, e = (float)(TILE - 1);
            const float umin = G0.delta + fminf(0.f, e * cc) + fminf(0.f, e * ss), umax = G0.delta + fmaxf(0.f, e * cc) + fmaxf(0.f, e * ss);
            const int tf = max(-1, (int)floorf((umin - a.margin + 0.5f) * 0.25f)), tl = min(FM_STRIPS - 2, (int)floorf((umax + a.margin + 0.5f) * 0.25f));
            s_t0[threadIdx.x] = (unsigned char)(tf + 1);
            s_tn[threadIdx.x] = (unsigned char)max(0, tl - tf + 1);
        }
        __syncthreads();
        if (threadIdx.x < 32) {                              // candidate table: pairs in order, their strips in order
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
            if (lane == 0) { s_ncand = base; s_nlong = 0; s_nshort = 0; s_next = 0; }
        }
        __syncthreads();
        // ---- work items: every candidate (pair, strip) is examined by one thread: the second angle's group of bins, the columns
        // the rays touch, and whether one 8-row window per column holds both angles (else one item per angle) ----
        for (int cnd = threadIdx.x; cnd < s_ncand; cnd += FM_THREADS) {
            const unsigned uu = s_cand[cnd];
            const FmPair R = s_pair[uu >> 4];
            const int ts = (int)(uu & 15) - 1;
            const float ft4 = 4.0f * (float)ts;
            int b1s = 0, cnt1 = 0;
            if (R.ib >= 0) {
                // angle-1 bin ub1 belongs to the strip whose extent [4 ts - 0.5, 4 ts + 3.5) holds phi(ub1): the extents tile the
                // line and both ends use the same expression, so every bin is in exactly one strip
                b1s = (int)ceilf((ft4 - 0.5f - R.r0) * R.rinv1);
                cnt1 = (int)ceilf((ft4 + 3.5f - R.r0) * R.rinv1) - b1s;
            }
            // first-tap row of window bin ub of angle x at column k:  (ub - delta) inv + k step
            const float y00 = (ft4 - R.delta0) * R.inv0, y03 = fmaf(3.0f, R.inv0, y00);
            const float y10 = ((float)b1s - R.delta1) * R.inv1, y11 = fmaf((float)(max(cnt1, 1) - 1), R.inv1, y10);
            const float lo0 = fminf(y00, y03), hi0 = fmaxf(y00, y03), lo1 = fminf(y10, y11), hi1 = fmaxf(y10, y11);
            int ka0, kb0, ka1 = TILE, kb1 = -1;
            col_range(lo0, hi0, R.step0, R.istep0, ka0, kb0);
            if (4 * ts + 3 < 0 || 4 * ts >= WIN) { ka0 = TILE; kb0 = -1; }          // no bin of the first angle's window in this strip
            if (cnt1 > 0 && b1s + cnt1 > 0 && b1s < WIN) col_range(lo1, hi1, R.step1, R.istep1, ka1, kb1);
            // one window for both angles?  The spread of first-tap rows is convex in k: check the two end columns
            bool pair_ok = cnt1 > 0 && cnt1 <= 4 && ka0 <= kb0 && ka1 <= kb1;
            if (pair_ok) {
                const float fa = (float)min(ka0, ka1), fb = (float)max(kb0, kb1);
                const float sa = fmaxf(fmaf(fa, R.step0, hi0), fmaf(fa, R.step1, hi1)) - fminf(fmaf(fa, R.step0, lo0), fmaf(fa, R.step1, lo1));
                const float sb = fmaxf(fmaf(fb, R.step0, hi0), fmaf(fb, R.step1, hi1)) - fminf(fmaf(fb, R.step0, lo0), fmaf(fb, R.step1, lo1));
                pair_ok = sa < FM_SPAN && sb < FM_SPAN;
            }
            // long items are handed out first (front of the list), short ones last (stored from the back): an even finish
            auto push = [&](const FmItem &x) {
                const bool lng = (int)x.khi - (int)x.klo >= FM_LONG;
                s_item[lng ? atomicAdd(&s_nlong, 1) : FM_MAXITEMS - 1 - atomicAdd(&s_nshort, 1)] = x;
            };
            FmItem it;
            it.pair_strip = (unsigned short)uu; it.b1s = (signed char)max(-100, min(100, b1s)); it.cnt1 = (unsigned char)min(cnt1, 8); it.pad = 0;
            if (pair_ok) {
                it.mode = 0; it.klo = (unsigned char)min(ka0, ka1); it.khi = (unsigned char)max(kb0, kb1);
                push(it);
            } else {
                if (ka0 <= kb0) { it.mode = 1; it.klo = (unsigned char)ka0; it.khi = (unsigned char)kb0; push(it); }
                if (ka1 <= kb1) { it.mode = 2; it.klo = (unsigned char)ka1; it.khi = (unsigned char)kb1; push(it); }
            }
        }
        __syncthreads();
        const int n_long = s_nlong, n_items = n_long + s_nshort;

        for (;;) {
            int u = 0;
            if (lane == 0) u = atomicAdd(&s_next, 1);
            u = __shfl_sync(0xffffffffu, u, 0);
            if (u >= n_items) break;
            const FmItem it = s_item[u < n_long ? u : FM_MAXITEMS - 1 - (u - n_long)];
            const FmPair R = s_pair[it.pair_strip >> 4];
            const int ts = (int)(it.pair_strip & 15) - 1, klo = it.klo, khi = it.khi, b1s = it.b1s, cnt1 = it.cnt1;
            // slot n of the 8 rays -> (angle, window bin).  mode 0: 0-3 first angle, 4-7 second; else one angle, slots from 0
            const bool use0 = it.mode != 2, use1 = it.mode != 1;
            const int off1 = it.mode == 0 ? 4 : 0;               // first slot of the second angle
            // lowest first-tap row of each angle in use at column 0: the window lines
            const float y00 = (4.0f * (float)ts - R.delta0) * R.inv0, y10 = ((float)b1s - R.delta1) * R.inv1;
            const float wl0 = use0 ? fminf(y00, fmaf(3.0f, R.inv0, y00)) : 1e6f;
            const float wl1 = use1 ? fminf(y10, fmaf((float)(max(cnt1, 1) - 1), R.inv1, y10)) : 1e6f;
            // my ray (slot g): B column g of the weight block, and the ray whose sums I add to P in the end
            const int bang = (use1 && !(use0 && g < 4)) ? 1 : 0;
            const int bub = bang ? b1s + g - off1 : 4 * ts + g;
            const bool bok = (bang ? (g >= off1 && g - off1 < cnt1) : (use0 && g < 4)) && bub >= 0 && bub < WIN;
            const float bstep = bang ? R.step1 : R.step0;
            // rows of column k0 at k = 2t, 2t+1 and of column k0+1 at k = 2t+8, 2t+9: first-tap row relative to row q + 2t
            const float byb = bok ? ((float)bub - (bang ? R.delta1 : R.delta0)) * (bang ? R.inv1 : R.inv0) - (float)(2 * t) : -1e6f;

            // window start per column: floor of the lowest first-tap row, clamped into the tile.  They are the same for every
            // lane, so lane s works out the pair of step s (columns kb + 2 s, kb + 2 s + 1) once per item and the loop fetches
            // it with one shuffle
            const int kb = klo & ~1;
            int qpack;
            {
                const float fk = (float)(kb + 2 * lane), fk1 = fk + 1.0f;
                const int qa = min(max((int)floorf(fminf(fmaf(fk, R.step0, wl0), fmaf(fk, R.step1, wl1))), 0), TILE - 8);
                const int qb = min(max((int)floorf(fminf(fmaf(fk1, R.step0, wl0), fmaf(fk1, R.step1, wl1))), 0), TILE - 8);
                qpack = qa | (qb << 8);
            }
            const float byb1 = byb + bstep;

            float acc[NB16][4];
#pragma unroll
            for (int zb = 0; zb < NB16; ++zb) acc[zb][0] = acc[zb][1] = acc[zb][2] = acc[zb][3] = 0.f;

            float fk = (float)kb;
            unsigned adr_k = ld_base + (unsigned)kb * (TILE * 16);
            const int nstep = ((khi - kb) >> 1) + 1;
            for (int st = 0; st < nstep; ++st, fk += 2.0f, adr_k += 2 * TILE * 16) {
                const int qp = __shfl_sync(0xffffffffu, qpack, st);
                const int qa = qp & 0xff, qb = qp >> 8;
                // weights of my ray at rows q + 2t, q + 2t + 1 of both columns: Joseph hat max(0, 1 - |row - y|)
                const float da = fmaf(fk, bstep, byb) - (float)qa, db = fmaf(fk, bstep, byb1) - (float)qb;   // y - (q + 2t)
                const float w0 = __saturatef(1.0f - fabsf(da)), w1 = __saturatef(1.0f - fabsf(da - 1.0f));
                const float w2 = __saturatef(1.0f - fabsf(db)), w3 = __saturatef(1.0f - fabsf(db - 1.0f));
                unsigned bh0, bl0, bh1, bl1;
                split2(w0, w1, bh0, bl0);
                split2(w2, w3, bh1, bl1);
                const unsigned adr = adr_k + ((unsigned)(ld_col ? qb : qa) << 4);
#pragma unroll
                for (int zb = 0; zb < NB16; ++zb) {
                    unsigned ah[4], al[4];
                    ldsm4t(ah, adr + zb * 2 * FM_PLANE);
                    ldsm4t(al, adr + zb * 2 * FM_PLANE + FM_PLANE);
                    mma16816(acc[zb], ah, bh0, bh1);
                    mma16816(acc[zb], al, bh0, bh1);
                    mma16816(acc[zb], ah, bl0, bl1);
                }
            }
            // ---- partial ray sums of this tile -> P[z][i][b][j].  My D entries are rays 2t, 2t+1 x batch entries g, g+8; a RED
            // costs about one clock per LANE whatever its width, so the block goes through a per-warp shared-memory patch and
            // leaves as one 16-byte RED per lane: lane (ray g, quad t) adds entries 4t .. 4t+3 of ray g ----
            const int i = bang ? R.ib : R.ia;
            const int b = (bang ? R.bstart1 : R.bstart0) + bub;
            const bool red_ok = bok && b >= 0 && b < a.nd;
            const float sc = bang ? R.inva1 : R.inva0;
#pragma unroll
            for (int zb = 0; zb < NB16; ++zb) {
                __syncwarp();
                stg[(2 * t) * FM_STG + g] = acc[zb][0];
                stg[(2 * t + 1) * FM_STG + g] = acc[zb][1];
                stg[(2 * t) * FM_STG + g + 8] = acc[zb][2];
                stg[(2 * t + 1) * FM_STG + g + 8] = acc[zb][3];
                __syncwarp();
                const float4 v = *reinterpret_cast<const float4 *>(stg + g * FM_STG + 4 * t);
                const int flat = zb * 16 + 4 * t, sl = z0 + (flat >> a.mshift), j = flat & (a.m - 1);
                if (red_ok && sl < a.nz)
                    atomicAdd(reinterpret_cast<float4 *>(P + (((int64_t)sl * a.n0 + i) * a.gp + a.gpl + b) * a.m + j),
                              make_float4(v.x * sc, v.y * sc, v.z * sc, v.w * sc));
            }
        }
    }
}

template <int NB16>
cudaError_t fm_launch(cp4d_ctx *c, const float *f, float *P, FmArgs a) {
    const Dims &d = c->d;
    a.zper = NB16 * 16 / d.m;
    const int zgroups = (d.nz + a.zper - 1) / a.zper;
    // small problems: split the angle pairs of a pass over up to 8 CTAs per tile so that every SM has work
    const int64_t ctas = (int64_t)d.tiles * 2 * zgroups;
    a.agroups = (int)std::max<int64_t>(1, std::min<int64_t>(std::min(8, std::max(1, std::min(c->n_pairs0, c->n_pairs1))), 148 / ctas));
    const dim3 grid(d.tiles * a.agroups, 2 * zgroups);
    k_forward_mma<NB16><<<grid, FM_THREADS, (size_t)NB16 * 2 * FM_PLANE, c->stream>>>(f, P, a);
    return cudaGetLastError();
}

}  // namespace

bool forward_mma_supported(const Dims &d) {
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

// host: pair adjacent base angles of one pass (same stepping axis, same sign of 1/ss, neighbouring indices); the angle with
// the smaller |1/ss| comes first, so that a strip of four of its bins holds at most four bins of the other
int forward_mma_pairs(const FwAngle *fw, const int32_t *order, int n0, int n_colstep, int2 *out, int *npairs0, int *npairs1) {
    int n = 0;
    // the second angle's rays are sorted into the first angle's strips by their position at the tile's middle column; a ray that
    // touches the tile is then at most 16 sqrt2 sin(pi/n0) bins outside the first angle's window, which the two spare strips
    // (bins -4 .. -1 and 48 .. 51) absorb for n0 >= 24.  Coarser angle sets run every angle on its own.
    const bool may_pair = n0 >= 24;
    for (int pass = 0; pass < 2; ++pass) {
        const int l0 = pass ? n_colstep : 0, l1 = pass ? n0 : n_colstep;
        const int start = n;
        for (int q = l0; q < l1;) {
            const int i = order[q];
            if (may_pair && q + 1 < l1 && order[q + 1] == i + 1 && (fw[i].inv > 0.f) == (fw[i + 1].inv > 0.f)) {
                const bool first = std::fabs(fw[i].inv) <= std::fabs(fw[i + 1].inv);
                out[n++] = first ? make_int2(i, i + 1) : make_int2(i + 1, i);
                q += 2;
            } else {
                out[n++] = make_int2(i, -1);
                q += 1;
            }
        }
        *(pass ? npairs1 : npairs0) = n - start;
    }
    return n;
}

cudaError_t launch_forward_mma(cp4d_ctx *c, const float *f, float *P) {
    const Dims &d = c->d;
    int ms = 0;
    while ((1 << ms) < d.m) ++ms;
    // 1.5 bins for the taps and the half-bin extents + (TILE/2) sqrt2 sin(pi/n0) for the drift over half a tile (pairs only)
    const float margin = 1.5f + (d.n0 >= 24 ? 0.5f * TILE * 1.41421356f * std::sin(3.14159265f / (float)d.n0) : 0.0f);
    FmArgs a{d.n, d.nz, d.nd, d.n0, d.m, ms, d.nd, 0, d.tiles, 1, 0, margin, c->geo, c->fwang, c->fw_pairs, c->n_pairs0, c->n_pairs1};
    // 16-entry batch blocks per CTA: three (192 KB of shared memory) unless the volume has fewer; m = 32 needs whole slices
    const int blocks_total = (d.nz * d.m + 15) / 16;
    int nb = std::min(3, blocks_total);
    if (d.m == 32) nb = 2;
    switch (nb) {
    case 1: return fm_launch<1>(c, f, P, a);
    case 2: return fm_launch<2>(c, f, P, a);
    default: return fm_launch<3>(c, f, P, a);
    }
}

}  // namespace cp4d
