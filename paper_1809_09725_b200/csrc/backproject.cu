// Adjoint projector, stage 2 (Eq. 10; fold L204-L212): backprojection of the pi-folded sinogram
// gt[z][i][jq][b] (float4 over 4 consecutive coefficients j) over the N_theta0 base angles.
//
// Operand delivery is what binds this kernel: shared memory hands out 32 lane-words/clk/SM, the FMA pipe
// eats 128 lanes/clk/SM.  So every fetched bin is reused from registers: a thread owns a compact PATCH of 2 (x) x 2 (y)
// voxels x 16 values (16 coefficients of one slice, 8 of two slices or 4 of four).  At one angle the patch touches only 4
// consecutive bins; they are loaded once (16 LDS.128) and feed 11 * 16 candidate FMAs, 8 * 16 of them real taps.
//
// Static register indexing.  With u = bin coordinate of a voxel, the patch's smallest coordinate is umin = K + phi
// (K integer, 0 <= phi < 1, both per thread) and voxel v sits at umin + delta_v where delta_v = e*|c| + dy*s is the
// same for every thread at this angle.  With an integer FL_v such that 0 <= delta_v - FL_v <= 1, t = phi + delta_v - FL_v is
// in [0,2) and the voxel touches only bins K+FL_v+{0,1,2}, with Joseph hat weights max(0, 1/a - |t-k|/a^2) (one of the three
// is zero): every register index is a compile-time constant.  For a 2 x 2 patch ONE tuple, FL = (0, 0, 0, 1), holds on all of
// [0, pi) (|c| + s >= 1), so there is no per-angle code selection (round 1's 4 x 2 patch needed 7 tuples and a switch).
// For c < 0 the patch is traversed mirrored in x (e = 1-dx): the staged chunks never mix the signs of c, and the accumulators
// are mirrored once, between the last chunk with c >= 0 and the first with c < 0.
#include <algorithm>
#include <cmath>

#include "cp4d_internal.cuh"
#include "device_helpers.cuh"

namespace cp4d {

namespace {

constexpr int WINP = WIN + 8;            // staged bins per (angle, row): window + spill, zero-filled outside the detector

// acc += w * v on 4 coefficients as two packed fp32x2 FMAs (SASS FFMA2: same FMA rate, half the issue slots)
__device__ __forceinline__ void fma4(float4 &a, const float2 ww, const float4 &v) {
    const float2 lo = __ffma2_rn(ww, make_float2(v.x, v.y), make_float2(a.x, a.y));
    const float2 hi = __ffma2_rn(ww, make_float2(v.z, v.w), make_float2(a.z, a.w));
    a = make_float4(lo.x, lo.y, hi.x, hi.y);
}
}  // namespace

struct BpArgs {
    int n, nz, nd, n0, Q, gp, gpl, n_pos;   // n_pos: the first n_pos base angles have c >= 0, the others c < 0
    int n_work;                             // work items = tiles * agroups * slice groups * coefficient groups
    int tiles, agroups;                     // item = tile + tiles * angle group (small grids split the base angles over CTAs,
                                            // which then ADD their partial sums to a zeroed output)
    const AngleTab *ang;
    const TileGeo *geo;
};

// ---------------------------------------------------------------------------------------------------
// k_backproject22<ZS>: 2 x 2 patches x 4 window rows per thread, a row = (slice, chunk of 4 coefficients): ZS = 1: four chunks
// of one slice (m % 16 == 0), ZS = 2: two chunks of two slices (m % 8 == 0), ZS = 4: one chunk of four slices.  The hat weights
// of a patch are computed once per angle and serve all four rows -- they do not depend on the slice or on the coefficient.
// 11 candidate FMAs for 8 taps; 4 bins x 4 rows = 16 LDS.128 per angle and thread.
// ---------------------------------------------------------------------------------------------------
constexpr int B22_THREADS = 256;         // one thread per 2 x 2 patch of a 32 x 32 tile
constexpr int B22_CHUNK = 15;            // angles staged per pipeline stage (2 stages x 15 x 4 rows of 896 B = 105 KB: two CTAs per SM)

// per (CTA, staged angle) parameters in shared memory, read by every thread as warp-uniform (broadcast) loads
struct B22Angle {
    float4 g;    // delta (tile origin - window start), c, s, |c|
    float4 k;    // A1 = 1/a, A2 = 1/a^2, A3 = A1 - 2 A2, |c| + s - 1
};

template <int ZS>
__global__ void __launch_bounds__(B22_THREADS, 2) k_backproject22(const float4 *__restrict__ gt, float *__restrict__ out, BpArgs a) {
    constexpr int QC = 4 / ZS;                                // coefficient chunks per slice; window row r = slice * QC + chunk
    extern __shared__ __align__(128) float4 win22[];          // [2][B22_CHUNK][4][WINP]
    __shared__ B22Angle sang[2][B22_CHUNK];
    __shared__ __align__(8) uint64_t mbar[2];
    const int tiles_1d = (a.n + TILE - 1) / TILE;
    const int per_z = a.tiles * a.agroups;
    const int wi = blockIdx.x;
    const int tile_id = (wi % per_z) % a.tiles, ag = (wi % per_z) / a.tiles;
    const int tix = tile_id % tiles_1d, tiy = tile_id / tiles_1d;
    const int nzg = (a.nz + ZS - 1) / ZS;
    const int z0 = ((wi / per_z) % nzg) * ZS, jg = wi / (per_z * nzg);    // ZS slices from z0, coefficient chunks jg QC .. jg QC + QC - 1
    const int zs_in = min(ZS, a.nz - z0);                                 // slices of this group inside the volume
    if (threadIdx.x == 0) {
        mbar_init(&mbar[0], 1);
        mbar_init(&mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    // lane -> patch: a quarter warp covers 2 (x) x 4 (y) patches; their window starts differ by at most 2|c| + 6 s < 6.4 slots of
    // 16 B, so the 8 lanes of an LDS.128 never collide on a bank
    const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int pxi = (l & 1) | ((l >> 3) << 1) | ((w & 1) << 3), pyi = ((l >> 1) & 3) | ((w >> 1) << 2);
    const float fx0 = (float)(2 * pxi), fy0 = (float)(2 * pyi);
    const TileGeo *geo = a.geo + (int64_t)tile_id * a.n0;
    const int g0 = (int)((int64_t)a.n0 * ag / a.agroups), g1 = (int)((int64_t)a.n0 * (ag + 1) / a.agroups);
    const int p0 = min(g0, a.n_pos), p1 = min(g1, a.n_pos), q0 = max(g0, a.n_pos), q1 = max(g1, a.n_pos);
    const int nchA = (p1 - p0 + B22_CHUNK - 1) / B22_CHUNK, nch = nchA + (q1 - q0 + B22_CHUNK - 1) / B22_CHUNK;
    auto chunk_begin = [&](int ch) { return ch < nchA ? p0 + ch * B22_CHUNK : q0 + (ch - nchA) * B22_CHUNK; };
    auto chunk_count = [&](int ch) { return min(B22_CHUNK, (ch < nchA ? p1 : q1) - chunk_begin(ch)); };
    auto stage = [&](int buf, int ch) {
        const int i0 = chunk_begin(ch), cnt = chunk_count(ch);
        if (threadIdx.x < B22_CHUNK) {
            const int i = min(i0 + (int)threadIdx.x, a.n0 - 1);
            const AngleTab A = a.ang[i];
            const float ca = fabsf(A.c), A2 = A.inv_a * A.inv_a;
            B22Angle &S = sang[buf][threadIdx.x];
            S.g = make_float4(geo[i].delta, A.c, A.s, ca);
            S.k = make_float4(A.inv_a, A2, fmaf(-2.0f, A2, A.inv_a), ca + A.s - 1.0f);
        }
        if (threadIdx.x < 32) {
            // rows of slices beyond the volume are not copied: their accumulators work on stale rows and are never stored
            if (threadIdx.x == 0) mbar_expect_tx(&mbar[buf], (unsigned)(cnt * zs_in * QC * WINP * sizeof(float4)));
            __syncwarp();
            for (int r = threadIdx.x; r < cnt * 4; r += 32) {
                const int aa = r >> 2, sl = (r & 3) / QC, jc = (r & 3) % QC, i = i0 + aa;
                if (sl < zs_in) {
                    const float4 *src = gt + (((int64_t)(z0 + sl) * a.n0 + i) * a.Q + jg * QC + jc) * a.gp + a.gpl + geo[i].bstart;
                    bulk_g2s(win22 + ((size_t)(buf * B22_CHUNK + aa) * 4 + (r & 3)) * WINP, src, (unsigned)(WINP * sizeof(float4)), &mbar[buf]);
                }
            }
        }
    };

    float4 acc[4][4];      // [voxel (e, dy) = (v & 1, v >> 1)][window row = (slice, coefficient chunk)]
#pragma unroll
    for (int v = 0; v < 4; ++v)
#pragma unroll
        for (int jc = 0; jc < 4; ++jc) acc[v][jc] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (nch > 0) stage(0, 0);
    __syncthreads();
    for (int ch = 0; ch < nch; ++ch) {
        const int buf = ch & 1;
        if (ch + 1 < nch) stage(buf ^ 1, ch + 1);
        mbar_wait(&mbar[buf], (ch >> 1) & 1);
        const int na = chunk_count(ch);
        const bool neg = ch >= nchA;
        if (ch == nchA) {            // from here on c < 0: the patch is traversed mirrored in x (e = 1 - dx)
#pragma unroll
            for (int dy = 0; dy < 2; ++dy)
#pragma unroll
                for (int jc = 0; jc < 4; ++jc) {
                    const float4 t0 = acc[2 * dy][jc]; acc[2 * dy][jc] = acc[2 * dy + 1][jc]; acc[2 * dy + 1][jc] = t0;
                }
        }
        for (int aa = 0; aa < na; ++aa) {
            const float4 G = sang[buf][aa].g, K = sang[buf][aa].k;
            const float umin = fmaf(fx0 + (neg ? 1.0f : 0.0f), G.y, fmaf(fy0, G.z, G.x));
            const float fk = floorf(umin), phi = umin - fk;
            // candidate weights max(0, 1/a - |t - k| / a^2), k = 0, 1, 2, of voxel v at t_v = phi + delta_v - FL_v in [0, 2)
            const float t1 = phi + G.w, t2 = phi + G.z, t3 = phi + K.w;
            const float w00 = fmaxf(0.f, fmaf(-K.y, phi, K.x)), w01 = fmaxf(0.f, fmaf(-K.y, 1.0f - phi, K.x));       // voxel 0: t < 1
            const float w10 = fmaxf(0.f, fmaf(-K.y, t1, K.x)), w11 = fmaxf(0.f, fmaf(-K.y, fabsf(t1 - 1.0f), K.x)), w12 = fmaxf(0.f, fmaf(K.y, t1, K.z));
            const float w20 = fmaxf(0.f, fmaf(-K.y, t2, K.x)), w21 = fmaxf(0.f, fmaf(-K.y, fabsf(t2 - 1.0f), K.x)), w22 = fmaxf(0.f, fmaf(K.y, t2, K.z));
            const float w30 = fmaxf(0.f, fmaf(-K.y, t3, K.x)), w31 = fmaxf(0.f, fmaf(-K.y, fabsf(t3 - 1.0f), K.x)), w32 = fmaxf(0.f, fmaf(K.y, t3, K.z));
            const float4 *wb = win22 + (size_t)(buf * B22_CHUNK + aa) * 4 * WINP + (int)fk;
#pragma unroll
            for (int jc = 0; jc < 4; ++jc) {
                const float4 b0 = wb[jc * WINP], b1 = wb[jc * WINP + 1], b2 = wb[jc * WINP + 2], b3 = wb[jc * WINP + 3];
                fma4(acc[0][jc], make_float2(w00, w00), b0); fma4(acc[0][jc], make_float2(w01, w01), b1);
                fma4(acc[1][jc], make_float2(w10, w10), b0); fma4(acc[1][jc], make_float2(w11, w11), b1); fma4(acc[1][jc], make_float2(w12, w12), b2);
                fma4(acc[2][jc], make_float2(w20, w20), b0); fma4(acc[2][jc], make_float2(w21, w21), b1); fma4(acc[2][jc], make_float2(w22, w22), b2);
                fma4(acc[3][jc], make_float2(w30, w30), b1); fma4(acc[3][jc], make_float2(w31, w31), b2); fma4(acc[3][jc], make_float2(w32, w32), b3);
            }
        }
        __syncthreads();
    }
    float4 *O = reinterpret_cast<float4 *>(out);
#pragma unroll
    for (int v = 0; v < 4; ++v) {
        const int x = tix * TILE + 2 * pxi + (nch > nchA ? 1 - (v & 1) : (v & 1)), y = tiy * TILE + 2 * pyi + (v >> 1);
        if (x < a.n && y < a.n) {
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                if (r / QC < zs_in) {
                    float4 *dst = O + (((int64_t)(z0 + r / QC) * a.n + y) * a.n + x) * a.Q + jg * QC + r % QC;
                    if (a.agroups == 1) *dst = acc[v][r];
                    else atomicAdd(dst, acc[v][r]);
                }
            }
        }
    }
}

template <int ZS>
static cudaError_t bp22_launch(cp4d_ctx *c, const float4 *gt, float *f_out, const BpArgs &a) {
    const Dims &d = c->d;
    constexpr int QC = 4 / ZS;
    const int64_t ctas = (int64_t)d.tiles * ((a.nz + ZS - 1) / ZS) * (a.Q / QC);
    BpArgs b = a;
    double best = 1e300;
    for (int ag = 1; ag <= std::min(8, d.n0); ++ag) {
        const int64_t waves = (ctas * ag + 148 * 2 - 1) / (148 * 2);
        const double cost = (double)waves * ((d.n0 + ag - 1) / ag + (ag > 1 ? 6 : 0));
        if (cost < best) { best = cost; b.agroups = ag; }
    }
    if (b.agroups > 1) {
        const cudaError_t e = cudaMemsetAsync(f_out, 0, (size_t)a.nz * d.n * d.n * a.Q * sizeof(float4), c->stream);
        if (e != cudaSuccess) return e;
        c->launches++;
    }
    b.n_work = (int)(ctas * b.agroups);
    k_backproject22<ZS><<<b.n_work, B22_THREADS, (size_t)2 * B22_CHUNK * 4 * WINP * sizeof(float4), c->stream>>>(gt, f_out, b);
    return cudaGetLastError();
}

cudaError_t backproject22_init() {
    constexpr int bytes = 2 * B22_CHUNK * 4 * WINP * (int)sizeof(float4);
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(k_backproject22<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(k_backproject22<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_backproject22<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

// Q_override > 0: backproject Q_override float4 chunks per bin / voxel instead of the context's Q (cp4d_fbp)
cudaError_t launch_backproject(cp4d_ctx *c, const float4 *gt, float *f_out, int Q_override) {
    ProfScope ps(c, CP4D_K_BACKPROJECT);
    const Dims &d = c->d;
    const int Q = Q_override > 0 ? Q_override : d.Q;
    BpArgs a{d.n, d.nz, d.nd, d.n0, Q, d.gp, d.gpl, c->n_cpos, 0, d.tiles, 1, c->ang, c->geo};
    c->launches++;
    if (Q % 4 == 0) return bp22_launch<1>(c, gt, f_out, a);
    if (Q % 2 == 0) return bp22_launch<2>(c, gt, f_out, a);
    return bp22_launch<4>(c, gt, f_out, a);
}

}  // namespace cp4d
