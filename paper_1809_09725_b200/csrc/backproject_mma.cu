// Adjoint projector on the tensor cores (Eq. 10; fold L204-L212): backprojection of the pi-folded sinogram over
// the base angles as small products  D[16 voxels x 8 batch entries] += W[16 voxels x 32 bins] * G[32 bins x 8]  with the
// weight block W as the 2:4 SPARSE operand of mma.sp (SASS HMMA.SP.16832) -- the transpose of forward_mma.cu, and the
// friendlier side of the pair:
//   * a 4 x 4 block of voxels touches at most 3 (|c| + |s|) + 3 <= 7.3 consecutive bins at ANY angle, so one 8-bin window per
//     angle holds every tap of the block: K = 32 = the 8-bin windows of four base angles (any four: no grouping condition),
//     M = 16 voxels = the block, and nothing is ever trimmed (100 % fill); a voxel's two taps at an angle are adjacent bins, so
//     every group of four bins of a window holds at most two of them -- the 2:4 structure;
//   * the accumulators are voxels: they stay in registers over all base angles and are written once -- no atomics.
// Operands are split bf16 pairs as in the forward kernel (G = Gh + Gl is written that way by k_fold_split, W = Wh + Wl per
// weight; D += Wh Gh + Wh Gl + Wl Gh, fp32 accumulation): relative error about 5e-6.
//
// CTA = (32 x 32 tile, group of NB16 16-entry batch blocks of (slice, coefficient)); warp w owns four 4 x 4 blocks.  The tile's
// bin windows of BM_STAGE base angles are staged by TMA 1-D bulk copies (SASS UBLKCP) into a two-stage ring: per angle and
// 8-entry half one copy of BM_WINP bins x 16 B out of the zero-padded rows of gt, so no bounds logic is needed.
#include <cuda_bf16.h>

#include <algorithm>
#include <cmath>

#include "cp4d_internal.cuh"
#include "device_helpers.cuh"

namespace cp4d {

namespace {

constexpr int BM_THREADS = 512;
constexpr int BM_STAGE = 8;                        // base angles per pipeline stage (a multiple of four: they are consumed four at a time)
constexpr int BM_WINP = 48;                        // staged bins per angle: a HALF tile (32 x 16 voxels) touches at most 31 |c| + 15 s + 3 < 38 bins,
                                                   // and any 8-bin window that starts among them is inside
constexpr int BM_HBLOCKS = (TILE / 4) * (TILE / 8);  // 4 x 4 voxel blocks of a half tile
constexpr int BM_BLOCKS = BM_HBLOCKS / (BM_THREADS / 32);               // 4 x 4 voxel blocks per warp

struct BmArgs {
    int n, nz, nd, n0, m, mshift, gp, gpl;
    int tiles, agroups;
    int zper;                                      // slices per CTA = NB16 * 16 / m
    const struct BmAngle *rec;                      // [tile][half][n0 + BM_STAGE] angle records, built once per context by k_bm_build
    const int *order;                               // tile of the i-th CTA of a launch row: bands of 8 tile rows, column by column
};

// per (tile, base angle): built once per context, staged by TMA (shared memory, broadcast loads)
struct BmAngle {
    float cmin;    // delta + min(0, 3c) + min(0, 3s): smallest window coordinate of a block is cmin + X0 c + Y0 s
    float delta, c, s;
    float A1, A2;  // Joseph hat in bin units, without its factor 1/a (k_fold_split applies it to the sinogram rows):
                   // weight(bin) = sat(A1 - A2 |u - bin|), A1 = 1, A2 = 1/a (0, 0 for an angle that weighs nothing)
    int bstart;    // first bin of the tile's window at this angle
    float pad;
};
static_assert(sizeof(BmAngle) == 32, "BmAngle is two 16-byte units");

// The angle records of every tile (they depend on the geometry only): n0 real ones and BM_STAGE that weigh nothing, so that the
// last stage of a CTA can always be staged whole.
__global__ void __launch_bounds__(128) k_bm_build(BmAngle *rec, const AngleTab *ang, const TileGeo *geo, int n0) {
    const int tile = blockIdx.x, half = blockIdx.y;
    for (int i = threadIdx.x; i < n0 + BM_STAGE; i += blockDim.x) {
        const int ii = min(i, n0 - 1);
        const AngleTab A = ang[ii];
        const TileGeo G = geo[(int64_t)tile * n0 + ii];
        // the lower half (rows 16 .. 31) starts 16 s further along the detector (s >= 0 on [0, pi)): its window starts floor(16 s)
        // bins later, and its coordinates are taken relative to its own first row
        const float off = 16.0f * (float)half * A.s, sh = floorf(off);
        BmAngle R;
        R.delta = G.delta + (off - sh);
        R.cmin = R.delta + fminf(0.f, 3.0f * A.c) + fminf(0.f, 3.0f * A.s);
        R.c = A.c; R.s = A.s;
        R.A1 = i < n0 ? 1.0f : 0.f; R.A2 = i < n0 ? A.inv_a : 0.f;
        R.bstart = G.bstart + (int)sh; R.pad = 0.f;
        rec[((int64_t)tile * 2 + half) * (n0 + BM_STAGE) + i] = R;
    }
}

// gt (split layout, written by k_fold_split): 16-byte units of 8 bf16 batch entries,
//   unit index = ((zg n0 + i) gp + gpl + b) U + hl H + half,  H = 2 NB16 halves per z-group, hl = 0 hi / 1 lo, U = 2 H + 1:
//   bin-major, so that the window of a tile at an angle is ONE contiguous run (one TMA copy per angle: the issue of a bulk copy
//   costs about 80 clk and holds up the other warps' shared-memory instructions, and 8 copies per angle were a fifth of the
//   kernel's time), and one unit of padding per bin, so that the 8 bins of an ldmatrix operand (stride U x 16 B) fall into 8
//   different bank groups
template <int NB16>
__global__ void __launch_bounds__(BM_THREADS, 1) k_backproject_mma(const uint4 *__restrict__ gt, float *__restrict__ out, BmArgs a) {
    constexpr int H = 2 * NB16;
    constexpr int U = 2 * H + 1;
    constexpr int ANGLE_UNITS = U * BM_WINP;                     // 16-byte units per staged angle: [bin][hl][half] + 1 of padding
    constexpr unsigned STAGE_BYTES = BM_STAGE * ANGLE_UNITS * 16;
    extern __shared__ __align__(128) unsigned char win[];         // [2 stages][BM_STAGE][BM_WINP][U] x 16 B
    __shared__ __align__(16) BmAngle sang[2][BM_STAGE];
    __shared__ __align__(4) unsigned char s_q[2][BM_HBLOCKS][BM_STAGE];                  // first bin of the 8-bin window of (block, angle)
    __shared__ __align__(8) uint64_t mbar[2];
    const int tiles_1d = (a.n + TILE - 1) / TILE;
    // CTAs that run at the same time should stage neighbouring windows (the folded sinogram of a z-group does not fit L2 at the
    // large configs): consecutive block indices walk the tiles in bands of 8 tile rows, column by column (a.order, host-made)
    const int ag = blockIdx.x / a.tiles, tile_id = a.order[blockIdx.x % a.tiles];
    const int zg = blockIdx.y, z0 = zg * a.zper, half = blockIdx.z;
    const int tx0 = (tile_id % tiles_1d) * TILE, ty0 = (tile_id / tiles_1d) * TILE + half * (TILE / 2);      // origin of my half tile
    const BmAngle *rec = a.rec + ((int64_t)tile_id * 2 + half) * (a.n0 + BM_STAGE);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, g = lane >> 2, t = lane & 3;
    // this CTA's share [g0, g1) of the base angles (small problems split them over CTAs, which then ADD into a zeroed output)
    const int g0 = (int)((int64_t)a.n0 * ag / a.agroups), g1 = (int)((int64_t)a.n0 * (ag + 1) / a.agroups);
    const int n_stage = (g1 - g0 + BM_STAGE - 1) / BM_STAGE;
    if (threadIdx.x == 0) {
        mbar_init(&mbar[0], 1);
        mbar_init(&mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();

    // Staging of stage st into buffer buf, so that no warp waits on global memory in the middle of its work:
    //   stage_issue (start of the previous stage's iteration, warp 0): one TMA copy of the stage's angle records and the TMA copies
    //     of the windows, whose row starts lanes < BM_STAGE loaded one call earlier (nb_bstart) and hand round by shuffle;
    //   stage_table (end of that iteration, warps < BM_STAGE): the window table of the stage from its records, which have landed
    //     long before (the mbarrier is still waited for: it orders the reads after the copies).
    int nb_bstart = 0;
    if (warp == 0 && lane < BM_STAGE) nb_bstart = rec[g0 + lane].bstart;
    auto stage_issue = [&](int buf, int st) {
        const int i0 = g0 + st * BM_STAGE;
        if (warp == 0) {
            if (lane == 0) {
                mbar_expect_tx(&mbar[buf], (unsigned)(BM_STAGE * ANGLE_UNITS * 16 + BM_STAGE * sizeof(BmAngle)));
                bulk_g2s(&sang[buf][0], rec + i0, (unsigned)(BM_STAGE * sizeof(BmAngle)), &mbar[buf]);
            }
            __syncwarp();
            if (lane < BM_STAGE) {                                     // one copy per angle
                const int i = min(i0 + lane, a.n0 - 1);
                const uint4 *src = gt + (((int64_t)zg * a.n0 + i) * a.gp + a.gpl + nb_bstart) * U;
                bulk_g2s(win + (size_t)buf * STAGE_BYTES + (size_t)lane * ANGLE_UNITS * 16, src, ANGLE_UNITS * 16, &mbar[buf]);
            }
            if (lane < BM_STAGE && st + 1 < n_stage) nb_bstart = rec[i0 + BM_STAGE + lane].bstart;      // used by the next call
        }
    };
    // 8-bin window of every (4 x 4 block, angle): from the smallest window coordinate of the block's 16 voxels; warp p fills angle p
    auto stage_table = [&](int buf, int st) {
        if (warp < BM_STAGE) {
            mbar_wait(&mbar[buf], (st >> 1) & 1);
            const BmAngle &S = sang[buf][warp];
            const float tc = S.c, ts = S.s, tcmin = S.cmin;
            const int bid = lane;                                      // BM_HBLOCKS = 32 blocks: one per lane
            const float u = fmaf((float)(4 * (bid & 7)), tc, fmaf((float)(4 * (bid >> 3)), ts, tcmin));
            s_q[buf][bid][warp] = (unsigned char)min(max((int)floorf(u), 0), BM_WINP - 8);
        }
    };

    float acc[BM_BLOCKS][NB16][2][4];     // [block][batch block][8-entry half]: voxels g (0, 1) and g + 8 (2, 3) x batch entries 2t, 2t + 1
#pragma unroll
    for (int q = 0; q < BM_BLOCKS; ++q)
#pragma unroll
        for (int zb = 0; zb < NB16; ++zb)
#pragma unroll
            for (int hf = 0; hf < 2; ++hf) acc[q][zb][hf][0] = acc[q][zb][hf][1] = acc[q][zb][hf][2] = acc[q][zb][hf][3] = 0.f;

    const unsigned win_s = smem_u32(win);
    // The weight block is the sparse operand: A[16 voxels x 32 bins], bin k = 8 aa + r = bin r of the 8-bin window of angle aa of
    // the group of four.  Lane (g, t) computes, for voxels g and g + 8 of the block ((g & 3, g >> 2) and two rows further), the
    // two kept elements of group t (angle t / 2, bins 4 (t & 1) .. + 3) and of group t + 4 (angle 2 + t / 2, same bins).
    const float vx = (float)(g & 3), vy = (float)(g >> 2);
    const int ka = t >> 1;                                           // my angles within the group: ka and ka + 2
    const float fh = (float)(4 * (t & 1));
    const unsigned qsel = 0x4440u + (unsigned)ka, qsel2 = qsel + 2u, msel = 0x4440u + (lane >> 3);
    if (n_stage > 0) { stage_issue(0, 0); stage_table(0, 0); }
    __syncthreads();
    for (int st = 0; st < n_stage; ++st) {
        const int buf = st & 1;
        // buffer buf^1 and sang[buf^1] were last read in the previous iteration, which ended with __syncthreads (s_q[buf^1] too:
        // it is rewritten at the end of this one)
        if (st + 1 < n_stage) stage_issue(buf ^ 1, st + 1);
        mbar_wait(&mbar[buf], (st >> 1) & 1);
#pragma unroll 1
        for (int p = 0; p < BM_STAGE; p += 4) {
            BmAngle S0 = sang[buf][p + ka], S1 = sang[buf][p + 2 + ka];
            // angles past this CTA's share (the tail of its last stage) weigh nothing
            if (g0 + st * BM_STAGE + p + ka >= g1) S0.A1 = S0.A2 = 0.f;
            if (g0 + st * BM_STAGE + p + 2 + ka >= g1) S1.A1 = S1.A2 = 0.f;
#pragma unroll
            for (int q = 0; q < BM_BLOCKS; ++q) {
                const int bid = warp * BM_BLOCKS + q;
                const float fx = (float)(4 * (bid & 7)) + vx, fy = (float)(4 * (bid >> 3)) + vy;
                const unsigned qw = *reinterpret_cast<const unsigned *>(&s_q[buf][bid][p]);      // window starts of the four angles
                const float fq0 = (float)__byte_perm(qw, 0u, qsel) + fh, fq1 = (float)__byte_perm(qw, 0u, qsel2) + fh;
                // window coordinate of my voxels relative to the first bin of my half window: voxel g, and g + 8 two rows further
                const float z00 = fmaf(fx, S0.c, fmaf(fy, S0.s, S0.delta)) - fq0, z01 = fmaf(2.0f, S0.s, z00);
                const float z10 = fmaf(fx, S1.c, fmaf(fy, S1.s, S1.delta)) - fq1, z11 = fmaf(2.0f, S1.s, z10);
                unsigned ah[4], al[4];
                float nib[4];
                auto kept = [&](float z, float A1, float A2, int slot) {
                    // the kept pair starts at bin i0 = clamp(floor(z), 0, 2) of the half window; positions (i0, i0 + 1), two bits each
                    const float i0 = fminf(fmaxf(floorf(z), 0.0f), 2.0f);
                    const float dd = z - i0;
                    nib[slot] = fmaf(5.0f, i0, 4.0f);
                    split2(__saturatef(fmaf(-A2, fabsf(dd), A1)), __saturatef(fmaf(-A2, fabsf(dd - 1.0f), A1)), ah[slot], al[slot]);
                };
                kept(z00, S0.A1, S0.A2, 0);      // a0: voxel g,     group t
                kept(z01, S0.A1, S0.A2, 1);      // a1: voxel g + 8, group t
                kept(z10, S1.A1, S1.A2, 2);      // a2: voxel g,     group t + 4
                kept(z11, S1.A1, S1.A2, 3);      // a3: voxel g + 8, group t + 4
                // metadata (device_helpers.cuh): lane 4g wants the groups 0-3 (low half: voxel g, high half: voxel g + 8), lane
                // 4g + 1 the groups 4-7; a butterfly over the quad
                unsigned e0 = (unsigned)__float2int_rn(fmaf(nib[1], 65536.0f, nib[0])) << (4 * t), e1 = (unsigned)__float2int_rn(fmaf(nib[3], 65536.0f, nib[2])) << (4 * t);
                e0 |= __shfl_xor_sync(0xffffffffu, e0, 2);
                e1 |= __shfl_xor_sync(0xffffffffu, e1, 2);
                const unsigned e = ((t & 1) ? e1 : e0) | __shfl_xor_sync(0xffffffffu, (t & 1) ? e0 : e1, 1);
                // ldmatrix: matrix = lane / 8 = angle of the group, row lane & 7 = bin of its window
                const unsigned adr = win_s + buf * STAGE_BYTES + (((p + (lane >> 3)) * BM_WINP + __byte_perm(qw, 0u, msel) + (lane & 7)) * (U * 16));
#pragma unroll
                for (int zb = 0; zb < NB16; ++zb)
#pragma unroll
                    for (int hf = 0; hf < 2; ++hf) {
                        unsigned bh[4], bl[4];
                        ldsm4t(bh, adr + (2 * zb + hf) * 16);
                        ldsm4t(bl, adr + (H + 2 * zb + hf) * 16);
                        mma_sp16832(acc[q][zb][hf], ah, bh, e);
                        mma_sp16832(acc[q][zb][hf], ah, bl, e);
                        mma_sp16832(acc[q][zb][hf], al, bh, e);
                    }
            }
        }
        if (st + 1 < n_stage) stage_table(buf ^ 1, st + 1);
        __syncthreads();
    }
    // ---- write the voxels: my D entries are voxels g, g + 8 of each block x batch entries 2t, 2t + 1 of each 8-entry half ----
#pragma unroll
    for (int q = 0; q < BM_BLOCKS; ++q) {
        const int bid = warp * BM_BLOCKS + q;
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            const int x = tx0 + 4 * (bid & 7) + (g & 3), y = ty0 + 4 * (bid >> 3) + (g >> 2) + 2 * r;
            if (x >= a.n || y >= a.n) continue;
#pragma unroll
            for (int zb = 0; zb < NB16; ++zb)
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    const int flat = zb * 16 + hf * 8 + 2 * t, sl = z0 + (flat >> a.mshift), j = flat & (a.m - 1);
                    if (sl >= a.nz) continue;
                    float *dst = out + (((int64_t)sl * a.n + y) * a.n + x) * a.m + j;
                    const float v0 = acc[q][zb][hf][2 * r], v1 = acc[q][zb][hf][2 * r + 1];
                    if (a.agroups == 1) *reinterpret_cast<float2 *>(dst) = make_float2(v0, v1);
                    else { atomicAdd(dst, v0); atomicAdd(dst + 1, v1); }
                }
        }
    }
}

// Fold for the tensor-core backprojector: gt_j[z][i][b] = sum_q Phi[j, q n0 + i] g[z][q n0 + i][flip_q b],
// written as split bf16 pairs in the layout k_backproject_mma stages.
template <int Q>
__global__ void __launch_bounds__(128) k_fold_split(const float *__restrict__ g, uint4 *__restrict__ gt, const float *__restrict__ phi,
                                                    int nd, int nz, int na, int npi, int n0, int gp, int gpl, int zper, int H, const AngleTab *__restrict__ ang) {
    extern __shared__ float phis[];  // [q][j], times the Joseph factor 1/a of the base angle (the backprojector's hat is normalised)
    // one CTA per (z-group, base angle i); thread = (bin, slice of the z-group), the slices of a bin in adjacent threads, so that
    // a bin's units (the 2 H hi / lo units of its U-unit record) are written by neighbouring lanes
    const int zg = blockIdx.x / n0, i = blockIdx.x % n0;
    constexpr int m = 4 * Q;
    const float inv_a = ang[i].inv_a;
    for (int t = threadIdx.x; t < npi * m; t += blockDim.x) phis[t] = phi[(int64_t)(t % m) * na + (t / m) * n0 + i] * inv_a;
    __syncthreads();
    const int sl = threadIdx.x % zper, z = zg * zper + sl, flat0 = sl * m;         // first batch entry of my slice inside its z-group
    const int U = 2 * H + 1;
    unsigned short *hi = reinterpret_cast<unsigned short *>(gt + ((int64_t)zg * n0 + i) * gp * U);
    unsigned short *lo = hi + H * 8;
    if (z >= nz) return;                                                            // (the scratch is zero there)
    for (int b = threadIdx.x / zper; b < nd; b += blockDim.x / zper) {
        float acc[m];
#pragma unroll
        for (int j = 0; j < m; ++j) acc[j] = 0.f;
        for (int q0 = 0; q0 < npi; q0 += 4) {     // 4 half-rotations per batch: their loads are in flight together
            float gv[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int q = min(q0 + u, npi - 1), bb = (q & 1) ? nd - 1 - b : b;
                gv[u] = __ldg(g + ((int64_t)z * na + q * n0 + i) * nd + bb);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (q0 + u < npi) {
#pragma unroll
                    for (int j = 0; j < m; ++j) acc[j] = fmaf(phis[(q0 + u) * m + j], gv[u], acc[j]);
                }
            }
        }
        // entries flat0 + j, j < m: 8-entry unit (flat0 + j) / 8 of the z-group, position (flat0 + j) % 8 -- whole 16-byte units
        // where the slice has 8 coefficients or more, runs of 4 otherwise
        if constexpr (Q >= 2) {
#pragma unroll
            for (int jc = 0; jc < Q; jc += 2) {
                const int flat = flat0 + 4 * jc;
                const int64_t e = ((int64_t)(gpl + b) * U + (flat >> 3)) * 8;
                uint4 h, l;
                split2(acc[4 * jc], acc[4 * jc + 1], h.x, l.x);
                split2(acc[4 * jc + 2], acc[4 * jc + 3], h.y, l.y);
                split2(acc[4 * jc + 4], acc[4 * jc + 5], h.z, l.z);
                split2(acc[4 * jc + 6], acc[4 * jc + 7], h.w, l.w);
                *reinterpret_cast<uint4 *>(hi + e) = h;
                *reinterpret_cast<uint4 *>(lo + e) = l;
            }
        } else {
            const int64_t e = ((int64_t)(gpl + b) * U + (flat0 >> 3)) * 8 + (flat0 & 7);
            unsigned h01, l01, h23, l23;
            split2(acc[0], acc[1], h01, l01);
            split2(acc[2], acc[3], h23, l23);
            *reinterpret_cast<uint2 *>(hi + e) = make_uint2(h01, h23);
            *reinterpret_cast<uint2 *>(lo + e) = make_uint2(l01, l23);
        }
    }
}

template <int NB16>
cudaError_t bm_launch(cp4d_ctx *c, const uint4 *gt, float *out, BmArgs a) {
    const Dims &d = c->d;
    a.zper = NB16 * 16 / d.m;
    const int zgroups = (d.nz + a.zper - 1) / a.zper;
    // small problems: split the base angles over up to 8 CTAs per tile, which add their partial sums into a zeroed output
    const int64_t ctas = (int64_t)d.tiles * 2 * zgroups;
    a.agroups = (int)std::max<int64_t>(1, std::min<int64_t>(std::min(8, std::max(1, d.n0 / BM_STAGE)), 148 / ctas));
    if (a.agroups > 1) {
        const cudaError_t e = cudaMemsetAsync(out, 0, (size_t)d.nz * d.n * d.n * d.m * sizeof(float), c->stream);
        if (e != cudaSuccess) return e;
        c->launches++;
    }
    const dim3 grid(d.tiles * a.agroups, zgroups, 2);
    k_backproject_mma<NB16><<<grid, BM_THREADS, (size_t)2 * BM_STAGE * (4 * NB16 + 1) * BM_WINP * 16, c->stream>>>(gt, out, a);
    return cudaGetLastError();
}

#define CP4D_BM_DISPATCH_Q(Qv, CALL)                       \
    switch (Qv) {                                          \
    case 1: { constexpr int QQ = 1; CALL; } break;         \
    case 2: { constexpr int QQ = 2; CALL; } break;         \
    case 4: { constexpr int QQ = 4; CALL; } break;         \
    default: { constexpr int QQ = 8; CALL; } break;        \
    }

}  // namespace

// 16-entry batch blocks per CTA of the tensor-core backprojector (also fixes the layout k_fold_split writes)
int backproject_mma_nb16(const Dims &d) {
    const int blocks_total = (d.nz * d.m + 15) / 16;
    return blocks_total >= 4 ? 4 : blocks_total >= 2 ? 2 : 1;      // (m = 32: the blocks of a slice come in pairs, so 2 or 4)
}

// 16-byte units of gt in the split layout (>= what the fp32 layout of the same scratch needs when nz is a multiple of zper)
int64_t backproject_mma_scratch_units(const Dims &d) {
    const int nb = backproject_mma_nb16(d), zper = nb * 16 / d.m, zgroups = (d.nz + zper - 1) / zper;
    return (int64_t)zgroups * d.n0 * (4 * nb + 1) * d.gp;
}

// bytes of the per-(tile, angle) records of a context (0 if the shape is not supported)
uint64_t backproject_mma_rec_bytes(const Dims &d) {
    return forward_mma_supported(d) ? (uint64_t)d.tiles * 2 * (d.n0 + BM_STAGE) * sizeof(BmAngle) : 0;
}

// host: the order in which a launch walks the tiles
void backproject_mma_order(int tiles_1d, int *order) {
    int k = 0;
    for (int band = 0; band * 8 < tiles_1d; ++band) {
        const int rows = std::min(8, tiles_1d - 8 * band);
        for (int tx = 0; tx < tiles_1d; ++tx)
            for (int r = 0; r < rows; ++r) order[k++] = (8 * band + r) * tiles_1d + tx;
    }
}

// cp4d_create: the angle records of every tile, once (they depend on the geometry only)
cudaError_t backproject_mma_build(cp4d_ctx *c) {
    if (!c->bm_rec) return cudaSuccess;
    k_bm_build<<<dim3(c->d.tiles, 2), 128, 0, c->stream>>>(reinterpret_cast<BmAngle *>(c->bm_rec), c->ang, c->geo, c->d.n0);
    return cudaGetLastError();
}

cudaError_t backproject_mma_init() {
    cudaError_t e = cudaFuncSetAttribute(k_backproject_mma<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * BM_STAGE * (4 * 1 + 1) * BM_WINP * 16);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_backproject_mma<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * BM_STAGE * (4 * 2 + 1) * BM_WINP * 16);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_backproject_mma<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * BM_STAGE * (4 * 4 + 1) * BM_WINP * 16);
}

cudaError_t launch_fold_split(cp4d_ctx *c, const float *g, float4 *gt) {
    ProfScope ps(c, CP4D_K_FOLD);
    const Dims &d = c->d;
    const int nb = backproject_mma_nb16(d), zper = nb * 16 / d.m;
    const size_t sh = (size_t)d.npi * d.m * sizeof(float);
    uint4 *G = reinterpret_cast<uint4 *>(gt);
    const int zgroups = (d.nz + zper - 1) / zper;
    CP4D_BM_DISPATCH_Q(d.Q, (k_fold_split<QQ><<<zgroups * d.n0, 128, sh, c->stream>>>(g, G, c->phi, d.nd, d.nz, d.na, d.npi, d.n0, d.gp, d.gpl, zper, 2 * nb, c->ang)));
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_backproject_mma(cp4d_ctx *c, const float4 *gt, float *f_out) {
    ProfScope ps(c, CP4D_K_BACKPROJECT);
    const Dims &d = c->d;
    int ms = 0;
    while ((1 << ms) < d.m) ++ms;
    BmArgs a{d.n, d.nz, d.nd, d.n0, d.m, ms, d.gp, d.gpl, d.tiles, 1, 0, reinterpret_cast<const BmAngle *>(c->bm_rec), c->bm_order};
    c->launches++;
    const uint4 *G = reinterpret_cast<const uint4 *>(gt);
    switch (backproject_mma_nb16(d)) {
    case 1: return bm_launch<1>(c, G, f_out, a);
    case 2: return bm_launch<2>(c, G, f_out, a);
    default: return bm_launch<4>(c, G, f_out, a);
    }
}

}  // namespace cp4d
