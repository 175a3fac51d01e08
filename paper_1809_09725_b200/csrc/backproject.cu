// Adjoint projector, stage 2 (Eq. 10; fold L204-L212): backprojection of the pi-folded sinogram
// gt[z][i][jq][b] (float4 over 4 consecutive coefficients j) over the N_theta0 base angles.
//
// Operand delivery is what binds this kernel: shared memory hands out 32 lane-words/clk/SM, the FMA pipe
// eats 128 lanes/clk/SM.  So every fetched bin is reused from registers: a thread owns a compact PATCH of 4 (x) x 2 (y)
// voxels x MJ = 4*JQ coefficients.  At one angle the patch touches only NB <= 6 consecutive bins; they are loaded once
// (NB*JQ LDS.128) and feed 16*MJ useful FMAs.
//
// Static register indexing.  With u = bin coordinate of a voxel, the patch's smallest coordinate is umin = K + phi
// (K integer, 0 <= phi < 1, both per thread) and voxel v sits at umin + delta_v where delta_v = e*|c| + dy*s is the
// same for every thread at this angle.  Choose an integer FL_v with 0 <= delta_v - FL_v <= 1 (the host picks one of
// 7 covering 8-tuples, the "pattern" of the angle); then t = phi + delta_v - FL_v is in [0,2) and the voxel touches only
// bins K+FL_v+{0,1,2}, with Joseph hat weights max(0, 1/a - |t-k|/a^2) (one of the three is zero).  A warp-uniform
// switch on the pattern selects straight-line code in which every register index is a compile-time constant.
// For c < 0 the patch is traversed mirrored in x (e = 3-dx): the staged chunks never mix the signs of c, and the accumulators
// are mirrored once, between the last chunk with c >= 0 and the first with c < 0.
#include <algorithm>
#include <cmath>

#include "cp4d_internal.cuh"
#include "device_helpers.cuh"

namespace cp4d {

namespace {

constexpr int BP_THREADS = 128;          // one thread per 4x2 patch of a 32x32 tile
constexpr int BP_CHUNK = 12;             // angles staged per pipeline stage
constexpr int WINP = WIN + 8;            // staged bins per (angle, jq): window + NB-1 spill, zero-filled outside the detector

__host__ __device__ constexpr int bp_fl(int pat, int v) {
    // 9 tuples floor(delta_v) occur over [0, pi); with the relaxed condition 0 <= delta_v - FL_v <= 1 these 7 cover every angle
    // (the tuples of theta = 0 and theta = pi/2 exactly are absorbed by their neighbours with an offset of exactly 1)
    constexpr int T[BP_NPAT][8] = {
        {0, 0, 1, 2, 0, 1, 2, 3}, {0, 0, 0, 0, 0, 1, 1, 1}, {0, 0, 1, 2, 0, 1, 2, 2}, {0, 0, 0, 1, 0, 1, 1, 2},
        {0, 0, 1, 1, 0, 1, 1, 2}, {0, 0, 1, 1, 0, 1, 2, 2}, {0, 0, 0, 1, 0, 1, 1, 1}};
    return T[pat][v];
}
__host__ __device__ constexpr int bp_nb(int pat) {
    int mx = 0;
    for (int v = 0; v < 8; ++v) mx = bp_fl(pat, v) > mx ? bp_fl(pat, v) : mx;
    return mx + 3;
}

// acc += w * v on 4 coefficients as two packed fp32x2 FMAs (SASS FFMA2: same FMA rate, half the issue slots)
__device__ __forceinline__ void fma4(float4 &a, const float2 ww, const float4 &v) {
    const float2 lo = __ffma2_rn(ww, make_float2(v.x, v.y), make_float2(a.x, a.y));
    const float2 hi = __ffma2_rn(ww, make_float2(v.z, v.w), make_float2(a.z, a.w));
    a = make_float4(lo.x, lo.y, hi.x, hi.y);
}
template <int PAT, int V, int JQ, int NB>
__device__ __forceinline__ void bp_voxel(float4 (&acc)[8][JQ], const float4 (&B)[NB][JQ], float phi, const float (&tdv)[8],
                                         float A1, float A2, float A3) {
    // accumulator V holds the voxel at offset (e, dy) = (V & 3, V >> 2) from the patch minimum: dx = e for c >= 0, dx = 3 - e
    // for c < 0 (the kernel mirrors the accumulators once when the sign of c changes)
    constexpr int E = V, FL = bp_fl(PAT, E);
    // E == 0 is the patch minimum itself: delta = 0, t = phi < 1, so its third candidate bin always has weight 0
    const float t = E == 0 ? phi : phi + tdv[E];                                  // in [0,2)
    const float x0 = fmaxf(0.f, fmaf(-A2, t, A1));
    const float x1 = fmaxf(0.f, fmaf(-A2, fabsf(t - 1.0f), A1));
    const float2 w0 = make_float2(x0, x0), w1 = make_float2(x1, x1);
#pragma unroll
    for (int jc = 0; jc < JQ; ++jc) {
        fma4(acc[V][jc], w0, B[FL][jc]);
        fma4(acc[V][jc], w1, B[FL + 1][jc]);
    }
    if (E != 0) {
        const float x2 = fmaxf(0.f, fmaf(A2, t, A3));                          // A3 = A1 - 2 A2
        const float2 w2 = make_float2(x2, x2);
#pragma unroll
        for (int jc = 0; jc < JQ; ++jc) fma4(acc[V][jc], w2, B[FL + 2][jc]);
    }
}

template <int PAT, int JQ>
__device__ __forceinline__ void bp_angle(float4 (&acc)[8][JQ], const float4 *wbase, float phi, const float4 tda,
                                         const float4 tdb, float A1, float A2, float A3) {
    constexpr int NB = bp_nb(PAT);
    float4 B[NB][JQ];
#pragma unroll
    for (int k = 0; k < NB; ++k)
#pragma unroll
        for (int jc = 0; jc < JQ; ++jc) B[k][jc] = wbase[jc * WINP + k];
    const float tdv[8] = {tda.x, tda.y, tda.z, tda.w, tdb.x, tdb.y, tdb.z, tdb.w};
    bp_voxel<PAT, 0, JQ, NB>(acc, B, phi, tdv, A1, A2, A3);
    bp_voxel<PAT, 1, JQ, NB>(acc, B, phi, tdv, A1, A2, A3);
    bp_voxel<PAT, 2, JQ, NB>(acc, B, phi, tdv, A1, A2, A3);
    bp_voxel<PAT, 3, JQ, NB>(acc, B, phi, tdv, A1, A2, A3);
    bp_voxel<PAT, 4, JQ, NB>(acc, B, phi, tdv, A1, A2, A3);
    bp_voxel<PAT, 5, JQ, NB>(acc, B, phi, tdv, A1, A2, A3);
    bp_voxel<PAT, 6, JQ, NB>(acc, B, phi, tdv, A1, A2, A3);
    bp_voxel<PAT, 7, JQ, NB>(acc, B, phi, tdv, A1, A2, A3);
}

}  // namespace

struct BpArgs {
    int n, nz, nd, n0, Q, gp, gpl, n_pos;   // n_pos: the first n_pos base angles have c >= 0, the others c < 0
    int n_work;                             // work items = tiles * agroups * nz * (Q / JQ)
    int tiles, agroups;                     // item = tile + tiles * angle group (small grids split the base angles over CTAs,
                                            // which then ADD their partial sums to a zeroed output)
    const AngleTab *ang;
    const TileGeo *geo;
};

// per (CTA, staged angle) parameters in shared memory, read by every thread as warp-uniform (broadcast) loads
struct BpAngle {
    float4 g;    // delta (tile origin - window start), c, s, unused
    float4 k;    // A1 = 1/a, A2 = 1/a^2, A3 = A1 - 2 A2, pattern (int bits)
    float4 tda;  // delta_v - FL_v for voxels v = 0..3 (dy = 0, e = 0..3)
    float4 tdb;  // v = 4..7 (dy = 1)
};

template <int JQ>
__global__ void __launch_bounds__(BP_THREADS, 4) k_backproject(const float4 *__restrict__ gt, float *__restrict__ out, BpArgs a) {
    __shared__ __align__(128) float4 win[2][BP_CHUNK][JQ][WINP];
    __shared__ BpAngle sang[2][BP_CHUNK];
    __shared__ __align__(8) uint64_t mbar[2];
    const int tiles_1d = (a.n + TILE - 1) / TILE;
    // work item w = (tile, angle group, slice, coefficient group), one CTA per item (the loop lets a smaller grid stride over them)
    const int per_z = a.tiles * a.agroups;
    unsigned cc = 0;                         // chunks staged so far by this CTA: buffer = cc & 1, mbarrier parity = (cc >> 1) & 1
    if (threadIdx.x == 0) {
        mbar_init(&mbar[0], 1);
        mbar_init(&mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    for (int wi = blockIdx.x; wi < a.n_work; wi += gridDim.x) {
    const int tile_id = (wi % per_z) % a.tiles, ag = (wi % per_z) / a.tiles;
    const int tix = tile_id % tiles_1d, tiy = tile_id / tiles_1d;
    const int z = (wi / per_z) % a.nz, jg = wi / (per_z * a.nz);
    // lane -> patch: a quarter warp (the unit an LDS.128 is served in) covers 2 (x) x 4 (y) patches; their window starts
    // differ by at most 4|c| + 6 s <= 7.2 < 8 slots of 16 B, so the 8 lanes never collide on a bank
    const int l = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int pxi = (l & 1) | ((l >> 2) & 6), pyi = ((l >> 1) & 3) | (w << 2);
    const float fx0 = (float)(4 * pxi), fy0 = (float)(2 * pyi);
    const TileGeo *geo = a.geo + (int64_t)tile_id * a.n0;
    // chunks never mix the signs of c: chunks of the angles with c >= 0 first, then of those with c < 0
    // this CTA's share [g0, g1) of the base angles, as its part [p0, p1) of those with c >= 0 and [q0, q1) of those with c < 0
    const int g0 = (int)((int64_t)a.n0 * ag / a.agroups), g1 = (int)((int64_t)a.n0 * (ag + 1) / a.agroups);
    const int p0 = min(g0, a.n_pos), p1 = min(g1, a.n_pos), q0 = max(g0, a.n_pos), q1 = max(g1, a.n_pos);
    const int nchA = (p1 - p0 + BP_CHUNK - 1) / BP_CHUNK, nch = nchA + (q1 - q0 + BP_CHUNK - 1) / BP_CHUNK;
    auto chunk_begin = [&](int ch) { return ch < nchA ? p0 + ch * BP_CHUNK : q0 + (ch - nchA) * BP_CHUNK; };
    auto chunk_count = [&](int ch) { return min(BP_CHUNK, (ch < nchA ? p1 : q1) - chunk_begin(ch)); };

    auto stage = [&](int buf, int ch) {
        const int i0 = chunk_begin(ch), cnt = chunk_count(ch);
        if (threadIdx.x < BP_CHUNK) {
            const int i = min(i0 + (int)threadIdx.x, a.n0 - 1);
            const AngleTab A = a.ang[i];
            const float ca = fabsf(A.c), A2 = A.inv_a * A.inv_a;
            float td[8];
#pragma unroll
            for (int v = 0; v < 8; ++v) td[v] = fmaf((float)(v & 3), ca, (float)(v >> 2) * A.s) - (float)((A.pat_fl >> (4 * v)) & 15);
            BpAngle &S = sang[buf][threadIdx.x];
            S.g = make_float4(geo[i].delta, A.c, A.s, 0.f);
            S.k = make_float4(A.inv_a, A2, fmaf(-2.0f, A2, A.inv_a), __int_as_float(A.pat));
            S.tda = make_float4(td[0], td[1], td[2], td[3]);
            S.tdb = make_float4(td[4], td[5], td[6], td[7]);
        }
        // one TMA bulk copy per (angle, coefficient chunk) row of the window: WINP bins x 16 B, always inside the padded
        // scratch row (cp4d_create checks), so no bounds logic; lanes 0..nrows-1 of warp 0 each issue one copy
        if (threadIdx.x < 32) {
            const int nrows = cnt * JQ;
            if (threadIdx.x == 0) mbar_expect_tx(&mbar[buf], (unsigned)(nrows * WINP * sizeof(float4)));
            __syncwarp();
            if ((int)threadIdx.x < nrows) {
                const int aa = threadIdx.x / JQ, jc = threadIdx.x % JQ, i = i0 + aa;
                const float4 *src = gt + (((int64_t)z * a.n0 + i) * a.Q + jg * JQ + jc) * a.gp + a.gpl + geo[i].bstart;
                bulk_g2s(&win[buf][aa][jc][0], src, (unsigned)(WINP * sizeof(float4)), &mbar[buf]);
            }
        }
    };

    float4 acc[8][JQ];
#pragma unroll
    for (int v = 0; v < 8; ++v)
#pragma unroll
        for (int jc = 0; jc < JQ; ++jc) acc[v][jc] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (nch > 0) stage((int)(cc & 1), 0);
    __syncthreads();
    for (int ch = 0; ch < nch; ++ch, ++cc) {
        const int buf = (int)(cc & 1);
        // buffer buf^1 and sang[buf^1] were last read in the previous chunk iteration, which ended with __syncthreads
        if (ch + 1 < nch) stage(buf ^ 1, ch + 1);
        mbar_wait(&mbar[buf], (cc >> 1) & 1);
        const int na = chunk_count(ch);
        // from the first chunk with c < 0 on, the patch is traversed mirrored in x (offset e = 3 - dx): swap the accumulators
        // once (warp-uniform, outside the angle loop) so that the same straight-line bodies serve both signs
        const bool neg = ch >= nchA;
        if (ch == nchA) {
#pragma unroll
            for (int dy = 0; dy < 2; ++dy)
#pragma unroll
                for (int jc = 0; jc < JQ; ++jc) {
                    const float4 t0 = acc[4 * dy + 0][jc]; acc[4 * dy + 0][jc] = acc[4 * dy + 3][jc]; acc[4 * dy + 3][jc] = t0;
                    const float4 t1 = acc[4 * dy + 1][jc]; acc[4 * dy + 1][jc] = acc[4 * dy + 2][jc]; acc[4 * dy + 2][jc] = t1;
                }
        }
        for (int aa = 0; aa < na; ++aa) {
            const BpAngle &S = sang[buf][aa];
            const float4 G = S.g, K = S.k;
            const float umin = fmaf(fx0 + (neg ? 3.0f : 0.0f), G.y, fmaf(fy0, G.z, G.x));
            const float fk = floorf(umin);
            const float phi = umin - fk;
            const float4 *wbase = &win[buf][aa][0][(int)fk];
            switch (__float_as_int(K.w)) {
            case 0: bp_angle<0, JQ>(acc, wbase, phi, S.tda, S.tdb, K.x, K.y, K.z); break;
            case 1: bp_angle<1, JQ>(acc, wbase, phi, S.tda, S.tdb, K.x, K.y, K.z); break;
            case 2: bp_angle<2, JQ>(acc, wbase, phi, S.tda, S.tdb, K.x, K.y, K.z); break;
            case 3: bp_angle<3, JQ>(acc, wbase, phi, S.tda, S.tdb, K.x, K.y, K.z); break;
            case 4: bp_angle<4, JQ>(acc, wbase, phi, S.tda, S.tdb, K.x, K.y, K.z); break;
            case 5: bp_angle<5, JQ>(acc, wbase, phi, S.tda, S.tdb, K.x, K.y, K.z); break;
            default: bp_angle<6, JQ>(acc, wbase, phi, S.tda, S.tdb, K.x, K.y, K.z); break;
            }
        }
        __syncthreads();
    }
    float4 *O = reinterpret_cast<float4 *>(out);
#pragma unroll
    for (int v = 0; v < 8; ++v) {
        const int x = tix * TILE + 4 * pxi + (nch > nchA ? 3 - (v & 3) : (v & 3)), y = tiy * TILE + 2 * pyi + (v >> 2);
        if (x < a.n && y < a.n) {
            float4 *dst = O + (((int64_t)z * a.n + y) * a.n + x) * a.Q + jg * JQ;
            if (a.agroups == 1) {
#pragma unroll
                for (int jc = 0; jc < JQ; ++jc) dst[jc] = acc[v][jc];
            } else {
#pragma unroll
                for (int jc = 0; jc < JQ; ++jc) atomicAdd(dst + jc, acc[v][jc]);
            }
        }
    }
    }   // work items
}

// ---------------------------------------------------------------------------------------------------
// 2 x 2 patches x 16 coefficients (m % 16 == 0): the hat weights of a patch are computed once per angle and serve all four
// coefficient chunks (the 4 x 2 kernel above computes them once per 8 coefficients), and ONE offset tuple serves every angle:
// with delta_v = e |c| + dy s the tuple FL = (0, 0, 0, 1) satisfies 0 <= delta_v - FL_v <= 1 on all of [0, pi) (|c| + s >= 1),
// so there is no pattern switch.  11 candidate FMAs for 8 taps (the 4 x 2 patch: 23 for 16).  The price is 4 bins x 4 chunks
// = 16 LDS.128 per angle and thread against 12 for twice the voxels.
// ---------------------------------------------------------------------------------------------------
constexpr int B22_THREADS = 256;         // one thread per 2 x 2 patch of a 32 x 32 tile
constexpr int B22_CHUNK = 15;            // angles staged per pipeline stage (2 stages x 15 x 4 rows of 896 B = 105 KB: two CTAs per SM)

struct B22Angle {
    float4 g;    // delta (tile origin - window start), c, s, |c|
    float4 k;    // A1 = 1/a, A2 = 1/a^2, A3 = A1 - 2 A2, |c| + s - 1
};

__global__ void __launch_bounds__(B22_THREADS, 2) k_backproject22(const float4 *__restrict__ gt, float *__restrict__ out, BpArgs a) {
    extern __shared__ __align__(128) float4 win22[];          // [2][B22_CHUNK][4][WINP]
    __shared__ B22Angle sang[2][B22_CHUNK];
    __shared__ __align__(8) uint64_t mbar[2];
    const int tiles_1d = (a.n + TILE - 1) / TILE;
    const int per_z = a.tiles * a.agroups;
    const int wi = blockIdx.x;
    const int tile_id = (wi % per_z) % a.tiles, ag = (wi % per_z) / a.tiles;
    const int tix = tile_id % tiles_1d, tiy = tile_id / tiles_1d;
    const int z = (wi / per_z) % a.nz, jg = wi / (per_z * a.nz);          // jg: group of 16 coefficients
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
            const int nrows = cnt * 4;
            if (threadIdx.x == 0) mbar_expect_tx(&mbar[buf], (unsigned)(nrows * WINP * sizeof(float4)));
            __syncwarp();
            for (int r = threadIdx.x; r < nrows; r += 32) {
                const int aa = r >> 2, jc = r & 3, i = i0 + aa;
                const float4 *src = gt + (((int64_t)z * a.n0 + i) * a.Q + jg * 4 + jc) * a.gp + a.gpl + geo[i].bstart;
                bulk_g2s(win22 + ((size_t)(buf * B22_CHUNK + aa) * 4 + jc) * WINP, src, (unsigned)(WINP * sizeof(float4)), &mbar[buf]);
            }
        }
    };

    float4 acc[4][4];      // [voxel (e, dy) = (v & 1, v >> 1)][coefficient chunk]
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
            float4 *dst = O + (((int64_t)z * a.n + y) * a.n + x) * a.Q + jg * 4;
#pragma unroll
            for (int jc = 0; jc < 4; ++jc) {
                if (a.agroups == 1) dst[jc] = acc[v][jc];
                else atomicAdd(dst + jc, acc[v][jc]);
            }
        }
    }
}

static cudaError_t bp22_launch(cp4d_ctx *c, const float4 *gt, float *f_out, const BpArgs &a) {
    const Dims &d = c->d;
    const int64_t ctas = (int64_t)d.tiles * a.nz * (a.Q / 4);
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
    k_backproject22<<<b.n_work, B22_THREADS, (size_t)2 * B22_CHUNK * 4 * WINP * sizeof(float4), c->stream>>>(gt, f_out, b);
    return cudaGetLastError();
}

cudaError_t backproject22_init() {
    return cudaFuncSetAttribute(k_backproject22, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * B22_CHUNK * 4 * WINP * (int)sizeof(float4));
}

template <int JQ>
static cudaError_t bp_launch(cp4d_ctx *c, const float4 *gt, float *f_out, const BpArgs &a) {
    const Dims &d = c->d;
    // small grids: whole waves of 148 SMs x 4 resident CTAs, least (waves x angles per CTA); the partial sums of the angle groups
    // are added into a zeroed output
    const int64_t ctas = (int64_t)d.tiles * a.nz * (a.Q / JQ);
    BpArgs b = a;
    double best = 1e300;
    for (int ag = 1; ag <= std::min(8, d.n0); ++ag) {
        const int64_t waves = (ctas * ag + 148 * 4 - 1) / (148 * 4);
        const double cost = (double)waves * ((d.n0 + ag - 1) / ag + (ag > 1 ? 6 : 0));
        if (cost < best) { best = cost; b.agroups = ag; }
    }
    if (b.agroups > 1) {
        const cudaError_t e = cudaMemsetAsync(f_out, 0, (size_t)a.nz * d.n * d.n * a.Q * sizeof(float4), c->stream);
        if (e != cudaSuccess) return e;
        c->launches++;
    }
    b.n_work = (int)(ctas * b.agroups);
    k_backproject<JQ><<<b.n_work, BP_THREADS, 0, c->stream>>>(gt, f_out, b);
    return cudaGetLastError();
}

// host side of the pattern choice (cp4d_create): first pattern whose offsets all satisfy 0 <= delta_v - FL_v <= 1,
// evaluated with the fp32-rounded |c|, s the kernel multiplies with
int bp_pattern(float c, float s) {
    const double ca = std::fabs((double)c), sd = (double)s;
    for (int p = 0; p < BP_NPAT; ++p) {
        bool ok = true;
        for (int v = 0; v < 8 && ok; ++v) {
            const double d = (v & 3) * ca + (v >> 2) * sd - bp_fl(p, v);
            ok = d >= 0.0 && d <= 1.0;
        }
        if (ok) return p;
    }
    return -1;
}

uint32_t bp_pattern_fl(int pat) {
    uint32_t r = 0;
    for (int v = 0; v < 8; ++v) r |= (uint32_t)bp_fl(pat, v) << (4 * v);
    return r;
}

// Q_override > 0: backproject Q_override float4 chunks per bin / voxel instead of the context's Q (cp4d_fbp)
cudaError_t launch_backproject(cp4d_ctx *c, const float4 *gt, float *f_out, int Q_override) {
    ProfScope ps(c, CP4D_K_BACKPROJECT);
    const Dims &d = c->d;
    const int Q = Q_override > 0 ? Q_override : d.Q;
    BpArgs a{d.n, d.nz, d.nd, d.n0, Q, d.gp, d.gpl, c->n_cpos, 0, d.tiles, 1, c->ang, c->geo};
    c->launches++;
    if (Q % 4 == 0) return bp22_launch(c, gt, f_out, a);      // 16 coefficients per thread: 3.77 -> 3.43 ms at config 3
    if (Q % 2 == 0) return bp_launch<2>(c, gt, f_out, a);
    return bp_launch<1>(c, gt, f_out, a);
}

}  // namespace cp4d
