// HBM-streaming kernels of the CP iteration (sm_100a): grad, div, the fused F2* prox (grad + projection,
// Fig. 2 step 4), the fused primal update (div + steps 5-6), the pi-fold prologue of the adjoint, the
// synthesis epilogue of the forward projector (optionally fused with the F1* prox, step 3), reductions.
//
// Layout f[z][iy][ix][j] (j fastest): one thread owns one float4 (4 consecutive coefficients j of one
// voxel) and walks along z, so the z neighbour is carried in registers and every 4D element is read
// from HBM once; x/y/t neighbours are served by L1/L2.  All global accesses are 16-byte, fully coalesced.
#include <algorithm>

#include "cp4d_internal.cuh"

namespace cp4d {

__device__ __forceinline__ float4 ld4(const float4 *p) { return __ldg(p); }
__device__ __forceinline__ float4 sub4(float4 a, float4 b) { return make_float4(a.x - b.x, a.y - b.y, a.z - b.z, a.w - b.w); }

// sum of v over the CTA, added to *slot (fp64)
__device__ __forceinline__ void block_add(double v, double *slot) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __shared__ double part[32];
    const int w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if ((threadIdx.x & 31) == 0) part[w] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int i = 0; i < nw; ++i) t += part[i];
        atomicAdd(slot, t);
    }
}

struct StreamArgs {
    int n, nz, Q, zper;
    int64_t slice4, V4;
    float lambda2;
    // z-slab contexts (cp4d_params.z_open): one read-only halo slice from the neighbour.
    //   k_grad: the slice of f above the slab (z = nz), so the z-difference of the last slice is not the boundary's 0;
    //   k_div:  the slice of p_z below the slab (z = -1); with hi_open the last slice's p_z is interior, not the boundary's 0
    const float4 *halo;
    int hi_open;
};

// ---------------------------------------------------------------------------------------------------
// MODE 0 grad:  p = K2 f.     MODE 1 prox: h2 <- proj_{|.|<=lambda1}(h2 + sigma K2 ft)
// MODE 2 tv:    *red += sum over (voxel, j) of |K2 f|_2   (the penalty of Eq. 6 without lambda1; nothing is stored)
// ---------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(256) k_grad(const float *__restrict__ f, float *__restrict__ p, StreamArgs a,
                                              float sigma, float inv_l1, int l1_zero, double *red) {
    const int64_t e4r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = e4r < a.slice4;
    if (MODE != 2 && !live) return;
    const int64_t e4 = live ? e4r : 0;   // MODE 2: idle threads still join the block reduction
    double tv = 0.0;
    const int c = (int)(e4 % a.Q);
    const int64_t vox = e4 / a.Q;
    const int x = (int)(vox % a.n), y = (int)(vox / a.n);
    const int z0 = blockIdx.y * a.zper, z1 = min(a.nz, z0 + a.zper);
    const float4 *F = reinterpret_cast<const float4 *>(f);
    float4 *P = reinterpret_cast<float4 *>(p);
    const bool hx = x + 1 < a.n, hy = y + 1 < a.n, ht = c + 1 < a.Q;
    const int64_t sy = (int64_t)a.n * a.Q;
    float4 cur = ld4(F + (int64_t)z0 * a.slice4 + e4);
    for (int z = z0; z < z1; ++z) {
        const int64_t idx = (int64_t)z * a.slice4 + e4;
        const float4 fz = (z + 1 < a.nz) ? ld4(F + idx + a.slice4) : (a.halo ? ld4(a.halo + e4) : cur);
        const float4 fx = hx ? ld4(F + idx + a.Q) : cur;
        const float4 fy = hy ? ld4(F + idx + sy) : cur;
        const float ft = ht ? __ldg(f + (idx + 1) * 4) : cur.w;
        float4 gx = sub4(fx, cur), gy = sub4(fy, cur), gz = sub4(fz, cur);
        float4 gt = make_float4(a.lambda2 * (cur.y - cur.x), a.lambda2 * (cur.z - cur.y), a.lambda2 * (cur.w - cur.z),
                                a.lambda2 * (ft - cur.w));
        if (MODE == 1) {
            float4 qx = P[idx], qy = P[idx + a.V4], qz = P[idx + 2 * a.V4], qt = P[idx + 3 * a.V4];
#define CP4D_PROX1(C)                                                                             \
    {                                                                                             \
        float vx = fmaf(sigma, gx.C, qx.C), vy = fmaf(sigma, gy.C, qy.C), vz = fmaf(sigma, gz.C, qz.C), \
              vt = fmaf(sigma, gt.C, qt.C);                                                       \
        float nn = sqrtf(fmaf(vx, vx, fmaf(vy, vy, fmaf(vz, vz, vt * vt))));                      \
        float r = l1_zero ? 0.0f : 1.0f / fmaxf(1.0f, nn * inv_l1);                               \
        gx.C = vx * r; gy.C = vy * r; gz.C = vz * r; gt.C = vt * r;                               \
    }
            CP4D_PROX1(x) CP4D_PROX1(y) CP4D_PROX1(z) CP4D_PROX1(w)
#undef CP4D_PROX1
        }
        if (MODE == 2) {
            if (live)
                tv += (double)sqrtf(gx.x * gx.x + gy.x * gy.x + gz.x * gz.x + gt.x * gt.x) +
                      (double)sqrtf(gx.y * gx.y + gy.y * gy.y + gz.y * gz.y + gt.y * gt.y) +
                      (double)sqrtf(gx.z * gx.z + gy.z * gy.z + gz.z * gz.z + gt.z * gt.z) +
                      (double)sqrtf(gx.w * gx.w + gy.w * gy.w + gz.w * gz.w + gt.w * gt.w);
        } else {
            P[idx] = gx;
            P[idx + a.V4] = gy;
            P[idx + 2 * a.V4] = gz;
            P[idx + 3 * a.V4] = gt;
        }
        cur = fz;
    }
    if (MODE == 2) block_add(tv, red);
}

// ---------------------------------------------------------------------------------------------------
// div (MODE 0): out = -K2^T p.
// update (MODE 1): f+ = f - tau bp + tau div h2; ft = f+ + theta (f+ - f); f <- f+   (steps 5-6)
// kkt (MODE 2): *red += sum (bp - div p)^2, nothing stored (bp = K1^T h1: the dual residual |K^T h|^2)
// ---------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(256) k_div(const float *__restrict__ p, float *__restrict__ out, StreamArgs a,
                                             const float *__restrict__ bp, float *__restrict__ ft_out, float tau,
                                             float theta, double *red) {
    const int64_t e4r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = e4r < a.slice4;
    if (MODE != 2 && !live) return;
    const int64_t e4 = live ? e4r : 0;
    double kk = 0.0;
    const int c = (int)(e4 % a.Q);
    const int64_t vox = e4 / a.Q;
    const int x = (int)(vox % a.n), y = (int)(vox / a.n);
    const int z0 = blockIdx.y * a.zper, z1 = min(a.nz, z0 + a.zper);
    const float4 *PX = reinterpret_cast<const float4 *>(p);
    const float4 *PY = PX + a.V4, *PZ = PX + 2 * a.V4, *PT = PX + 3 * a.V4;
    const float *pt_s = p + 3 * a.V4 * 4;
    const int64_t sy = (int64_t)a.n * a.Q;
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
    float4 prevz = (z0 > 0) ? ld4(PZ + (int64_t)(z0 - 1) * a.slice4 + e4) : (a.halo ? ld4(a.halo + e4) : zero);
    for (int z = z0; z < z1; ++z) {
        const int64_t idx = (int64_t)z * a.slice4 + e4;
        const float4 xc = (x < a.n - 1) ? ld4(PX + idx) : zero;
        const float4 xm = (x > 0) ? ld4(PX + idx - a.Q) : zero;
        const float4 yc = (y < a.n - 1) ? ld4(PY + idx) : zero;
        const float4 ym = (y > 0) ? ld4(PY + idx - sy) : zero;
        const float4 zc = (z < a.nz - 1 || a.hi_open) ? ld4(PZ + idx) : zero;
        const float4 tc = ld4(PT + idx);
        const float tm = (c > 0) ? __ldg(pt_s + idx * 4 - 1) : 0.0f;
        const float tw = (c < a.Q - 1) ? tc.w : 0.0f;
        float4 d;
        d.x = (xc.x - xm.x) + (yc.x - ym.x) + (zc.x - prevz.x) + a.lambda2 * (tc.x - tm);
        d.y = (xc.y - xm.y) + (yc.y - ym.y) + (zc.y - prevz.y) + a.lambda2 * (tc.y - tc.x);
        d.z = (xc.z - xm.z) + (yc.z - ym.z) + (zc.z - prevz.z) + a.lambda2 * (tc.z - tc.y);
        d.w = (xc.w - xm.w) + (yc.w - ym.w) + (zc.w - prevz.w) + a.lambda2 * (tw - tc.z);
        if (MODE == 2) {
            const float4 b = ld4(reinterpret_cast<const float4 *>(bp) + idx);
            const float ex = b.x - d.x, ey = b.y - d.y, ez = b.z - d.z, ew = b.w - d.w;
            if (live) kk += (double)ex * ex + (double)ey * ey + (double)ez * ez + (double)ew * ew;
        } else if (MODE == 1) {
            float4 *F = reinterpret_cast<float4 *>(out);
            const float4 fo = F[idx];
            const float4 b = ld4(reinterpret_cast<const float4 *>(bp) + idx);
            float4 fn, fr;
            fn.x = fmaf(tau, d.x - b.x, fo.x); fn.y = fmaf(tau, d.y - b.y, fo.y);
            fn.z = fmaf(tau, d.z - b.z, fo.z); fn.w = fmaf(tau, d.w - b.w, fo.w);
            fr.x = fmaf(theta, fn.x - fo.x, fn.x); fr.y = fmaf(theta, fn.y - fo.y, fn.y);
            fr.z = fmaf(theta, fn.z - fo.z, fn.z); fr.w = fmaf(theta, fn.w - fo.w, fn.w);
            F[idx] = fn;
            reinterpret_cast<float4 *>(ft_out)[idx] = fr;
        } else {
            reinterpret_cast<float4 *>(out)[idx] = d;
        }
        prevz = zc;
    }
    if (MODE == 2) block_add(kk, red);
}

static StreamArgs make_args(const cp4d_ctx *c, dim3 &grid, dim3 &block, const float *halo = nullptr) {
    const Dims &d = c->d;
    StreamArgs a;
    a.n = d.n; a.nz = d.nz; a.Q = d.Qp; a.slice4 = d.slice4; a.V4 = d.V / 4; a.lambda2 = c->lambda2;
    a.halo = reinterpret_cast<const float4 *>(halo); a.hi_open = (c->z_open & 2) ? 1 : 0;
    block = dim3(256);
    const int64_t bx = (d.slice4 + 255) / 256;
    // enough CTAs to fill 148 SMs x 8 resident CTAs a few times over; otherwise split z
    int zchunks = 1;
    while (bx * zchunks < 148 * 16 && zchunks < d.nz) zchunks *= 2;
    if (zchunks > d.nz) zchunks = d.nz;
    a.zper = (d.nz + zchunks - 1) / zchunks;
    grid = dim3((unsigned)bx, (unsigned)((d.nz + a.zper - 1) / a.zper));
    return a;
}

cudaError_t launch_grad(cp4d_ctx *c, const float *f, float *p, const float *halo) {
    ProfScope ps(c, CP4D_K_GRAD);
    dim3 g, b;
    StreamArgs a = make_args(c, g, b, halo);
    k_grad<0><<<g, b, 0, c->stream>>>(f, p, a, 0.f, 0.f, 0, nullptr);
    c->launches++;
    return cudaGetLastError();
}
cudaError_t launch_prox_f2(cp4d_ctx *c, float sigma, const float *ft, float *h2, const float *halo) {
    ProfScope ps(c, CP4D_K_PROX_F2);
    dim3 g, b;
    StreamArgs a = make_args(c, g, b, halo);
    const int l1z = !(c->lambda1 > 0.f);
    k_grad<1><<<g, b, 0, c->stream>>>(ft, h2, a, sigma, l1z ? 0.f : 1.0f / c->lambda1, l1z, nullptr);
    c->launches++;
    return cudaGetLastError();
}
cudaError_t launch_div(cp4d_ctx *c, const float *p, float *f, const float *halo) {
    ProfScope ps(c, CP4D_K_DIV);
    dim3 g, b;
    StreamArgs a = make_args(c, g, b, halo);
    k_div<0><<<g, b, 0, c->stream>>>(p, f, a, nullptr, nullptr, 0.f, 0.f, nullptr);
    c->launches++;
    return cudaGetLastError();
}
cudaError_t launch_update(cp4d_ctx *c, float tau, const float *bp, const float *h2, float *f, float *ft, const float *halo) {
    ProfScope ps(c, CP4D_K_UPDATE);
    dim3 g, b;
    StreamArgs a = make_args(c, g, b, halo);
    k_div<1><<<g, b, 0, c->stream>>>(h2, f, a, bp, ft, tau, c->theta, nullptr);
    c->launches++;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------
// frame <-> coefficient contraction per voxel:  out[v][a] = sum_b T(a,b) in[v][b]
//   analysis     f_j = sum_q phi_j(t_q) f(t_q):  a = j, b = q;   its transpose (after K1^T):  a = q, b = j
// One thread per (voxel, 4 outputs); T sits in shared memory as Tt[b][a]; HBM-bound (reads NB, writes NA floats per voxel).
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_mix(const float4 *__restrict__ in, float4 *__restrict__ out, const float *__restrict__ psi,
                                             int64_t nvox, int QA, int QB, int sa, int sb) {
    extern __shared__ float Tt[];  // [NB][NA]
    const int NA = 4 * QA, NB = 4 * QB;
    for (int t = threadIdx.x; t < NA * NB; t += blockDim.x) {
        const int b = t / NA, a = t % NA;
        Tt[t] = psi[a * sa + b * sb];
    }
    __syncthreads();
    const int64_t total = nvox * QA, stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += stride) {
        const int64_t v = e / QA;
        const int ca = (int)(e % QA);
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        const float4 *row = in + v * QB;
        for (int bc = 0; bc < QB; ++bc) {
            const float4 x = ld4(row + bc);
            const float4 *T4 = reinterpret_cast<const float4 *>(Tt + (4 * bc) * NA + 4 * ca);
            const float4 t0 = T4[0], t1 = T4[NA / 4], t2 = T4[2 * (NA / 4)], t3 = T4[3 * (NA / 4)];
            acc.x = fmaf(t0.x, x.x, fmaf(t1.x, x.y, fmaf(t2.x, x.z, fmaf(t3.x, x.w, acc.x))));
            acc.y = fmaf(t0.y, x.x, fmaf(t1.y, x.y, fmaf(t2.y, x.z, fmaf(t3.y, x.w, acc.y))));
            acc.z = fmaf(t0.z, x.x, fmaf(t1.z, x.y, fmaf(t2.z, x.z, fmaf(t3.z, x.w, acc.z))));
            acc.w = fmaf(t0.w, x.x, fmaf(t1.w, x.y, fmaf(t2.w, x.z, fmaf(t3.w, x.w, acc.w))));
        }
        out[e] = acc;
    }
}

cudaError_t launch_mix(cp4d_ctx *c, const float *in, float *out, int na_out, int nb_in, int sa, int sb) {
    ProfScope ps(c, CP4D_K_MIX);
    const Dims &d = c->d;
    const int64_t nvox = (int64_t)d.nz * d.n * d.n;
    const int64_t total = nvox * (na_out / 4);
    const int64_t blocks = std::min<int64_t>((total + 255) / 256, 148 * 16);   // grid-stride: Psi is staged once per CTA
    k_mix<<<(unsigned)blocks, 256, (size_t)na_out * nb_in * sizeof(float), c->stream>>>(
        reinterpret_cast<const float4 *>(in), reinterpret_cast<float4 *>(out), c->psi, nvox, na_out / 4, nb_in / 4, sa, sb);
    c->launches++;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------
// static FBP per half-rotation
// ---------------------------------------------------------------------------------------------------
// Shepp-Logan filter, unit bin spacing, direct convolution:  gf[b] = sum_b' h[b-b'] g[b'],  h[n] = -2 / (pi^2 (4 n^2 - 1)).
// One CTA per sinogram row (z, k); the row sits in shared memory.
__global__ void __launch_bounds__(256) k_filter_sl(const float *__restrict__ g, float *__restrict__ gf, int nd) {
    extern __shared__ float row[];
    const float *src = g + (int64_t)blockIdx.x * nd;
    for (int b = threadIdx.x; b < nd; b += blockDim.x) row[b] = __ldg(src + b);
    __syncthreads();
    const float k0 = -0.20264236728467555f;   // -2 / pi^2
    for (int b = threadIdx.x; b < nd; b += blockDim.x) {
        float acc = 0.f;
        for (int bp = 0; bp < nd; ++bp) {
            const float n = (float)(b - bp);
            acc = fmaf(__fdividef(k0, fmaf(4.0f * n, n, -1.0f)), row[bp], acc);
        }
        gf[(int64_t)blockIdx.x * nd + b] = acc;
    }
}
cudaError_t launch_filter_sl(cp4d_ctx *c, const float *g, float *gf) {
    ProfScope ps(c, CP4D_K_MISC);
    const Dims &d = c->d;
    k_filter_sl<<<(unsigned)(d.nz * d.na), 256, (size_t)d.nd * sizeof(float), c->stream>>>(g, gf, d.nd);
    c->launches++;
    return cudaGetLastError();
}
// gt[z][i][qc][gpl + b] = scale * (gf[z][q n0 + i][flip_q b])_{q = 4 qc .. 4 qc + 3}: the fold with the box basis
// phi_q = 1 on half-rotation q, whose backprojection is the static reconstruction of every half-rotation at once
__global__ void __launch_bounds__(128) k_fold_halfrot(const float *__restrict__ gf, float4 *__restrict__ gt, int nd, int na, int npi,
                                                     int n0, int gp, int gpl, int Qf, float scale) {
    const int z = blockIdx.x / n0, i = blockIdx.x % n0;
    for (int t = threadIdx.x; t < Qf * nd; t += blockDim.x) {
        const int qc = t / nd, b = t % nd;
        float v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int q = 4 * qc + u;
            v[u] = q < npi ? scale * __ldg(gf + ((int64_t)z * na + q * n0 + i) * nd + ((q & 1) ? nd - 1 - b : b)) : 0.f;
        }
        gt[(((int64_t)z * n0 + i) * Qf + qc) * gp + gpl + b] = make_float4(v[0], v[1], v[2], v[3]);
    }
}
cudaError_t launch_fold_halfrot(cp4d_ctx *c, const float *gf, float4 *gt, int Qf, float scale) {
    ProfScope ps(c, CP4D_K_FOLD);
    const Dims &d = c->d;
    k_fold_halfrot<<<d.nz * d.n0, 128, 0, c->stream>>>(gf, gt, d.nd, d.na, d.npi, d.n0, d.gp, d.gpl, Qf, scale);
    c->launches++;
    return cudaGetLastError();
}

// reductions for cp4d_objective: *slot is zeroed first, then accumulated by the kernel
cudaError_t launch_tv_sum(cp4d_ctx *c, const float *f, double *slot) {
    ProfScope ps(c, CP4D_K_REDUCE);
    dim3 g, b;
    StreamArgs a = make_args(c, g, b);
    cudaError_t e = cudaMemsetAsync(slot, 0, sizeof(double), c->stream);
    if (e != cudaSuccess) return e;
    k_grad<2><<<g, b, 0, c->stream>>>(f, nullptr, a, 0.f, 0.f, 0, slot);
    c->launches += 2;
    return cudaGetLastError();
}
cudaError_t launch_kkt_sum(cp4d_ctx *c, const float *bp, const float *h2, double *slot) {
    ProfScope ps(c, CP4D_K_REDUCE);
    dim3 g, b;
    StreamArgs a = make_args(c, g, b);
    cudaError_t e = cudaMemsetAsync(slot, 0, sizeof(double), c->stream);
    if (e != cudaSuccess) return e;
    k_div<2><<<g, b, 0, c->stream>>>(h2, nullptr, a, bp, nullptr, 0.f, 0.f, slot);
    c->launches += 2;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------
// fold: gt[z][i][jc][b] (float4 over j) = sum_q Phi[j, q n0 + i] g[z][q n0 + i][flip_q b]
// synth (PAPER.md:L198-L202 + Eq. 9): v[z][q n0+i][flip_q b] = sum_j Phi[j, q n0+i] P[z][i][b][j]   (P: j fastest, row pitch gp bins)
// One CTA per (z, base angle i); the npi x m slice of Phi it needs sits in shared memory.
// ---------------------------------------------------------------------------------------------------
template <int Q>
__global__ void __launch_bounds__(128) k_fold(const float *__restrict__ g, float4 *__restrict__ gt,
                                              const float *__restrict__ phi, int nd, int na, int npi, int n0, int gp, int gpl) {
    extern __shared__ float phis[];  // [q][j]
    const int z = blockIdx.x / n0, i = blockIdx.x % n0;
    constexpr int m = 4 * Q;
    for (int t = threadIdx.x; t < npi * m; t += blockDim.x) phis[t] = phi[(int64_t)(t % m) * na + (t / m) * n0 + i];
    __syncthreads();
    for (int b = threadIdx.x; b < nd; b += blockDim.x) {
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
#pragma unroll
        for (int jc = 0; jc < Q; ++jc)
            gt[(((int64_t)z * n0 + i) * Q + jc) * gp + gpl + b] = make_float4(acc[4 * jc], acc[4 * jc + 1], acc[4 * jc + 2], acc[4 * jc + 3]);
    }
}

template <int Q>
__global__ void __launch_bounds__(128) k_synth(const float4 *__restrict__ P, int mode, float sigma,
                                               const float *__restrict__ g, float *__restrict__ out,
                                               const float *__restrict__ phi, const FwAngle *__restrict__ fwang, int nd, int na, int npi,
                                               int n0, int gp, int gpl) {
    extern __shared__ float phis[];
    const int z = blockIdx.x / n0, i = blockIdx.x % n0;
    constexpr int m = 4 * Q;
    // the projectors leave P without the Joseph normalisation 1/max(|c|,|s|) of its base angle: it is folded into Phi here
    const float inv_a = fwang[i].inv_a;
    for (int t = threadIdx.x; t < npi * m; t += blockDim.x) phis[t] = phi[(int64_t)(t % m) * na + (t / m) * n0 + i] * inv_a;
    __syncthreads();
    const float rs = 1.0f / (1.0f + sigma);
    for (int b = threadIdx.x; b < nd; b += blockDim.x) {
        float acc[m];
#pragma unroll
        for (int jc = 0; jc < Q; ++jc) {
            const float4 v = P[(((int64_t)z * n0 + i) * gp + gpl + b) * Q + jc];
            acc[4 * jc] = v.x; acc[4 * jc + 1] = v.y; acc[4 * jc + 2] = v.z; acc[4 * jc + 3] = v.w;
        }
        for (int q0 = 0; q0 < npi; q0 += 4) {     // 4 half-rotations per batch: their loads are in flight together
            float ho[4], gg[4];
            int64_t idx[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int q = min(q0 + u, npi - 1), bb = (q & 1) ? nd - 1 - b : b;
                idx[u] = ((int64_t)z * na + q * n0 + i) * nd + bb;
                if (mode != 0) { ho[u] = out[idx[u]]; gg[u] = __ldg(g + idx[u]); }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (q0 + u < npi) {
                    float v = 0.f;
#pragma unroll
                    for (int j = 0; j < m; ++j) v = fmaf(phis[(q0 + u) * m + j], acc[j], v);
                    out[idx[u]] = (mode == 0) ? v : (ho[u] + sigma * (v - gg[u])) * rs;
                }
            }
        }
    }
}

#define CP4D_DISPATCH_Q(Qv, CALL)                          \
    switch (Qv) {                                          \
    case 1: { constexpr int QQ = 1; CALL; } break;         \
    case 2: { constexpr int QQ = 2; CALL; } break;         \
    case 3: { constexpr int QQ = 3; CALL; } break;         \
    case 4: { constexpr int QQ = 4; CALL; } break;         \
    case 5: { constexpr int QQ = 5; CALL; } break;         \
    case 6: { constexpr int QQ = 6; CALL; } break;         \
    case 7: { constexpr int QQ = 7; CALL; } break;         \
    default: { constexpr int QQ = 8; CALL; } break;        \
    }

cudaError_t launch_fold(cp4d_ctx *c, const float *g, float4 *gt) {
    ProfScope ps(c, CP4D_K_FOLD);
    const Dims &d = c->d;
    const size_t sh = (size_t)d.npi * d.m * sizeof(float);
    CP4D_DISPATCH_Q(d.Q, (k_fold<QQ><<<d.nz * d.n0, 128, sh, c->stream>>>(g, gt, c->phi, d.nd, d.na, d.npi, d.n0, d.gp, d.gpl)));
    c->launches++;
    return cudaGetLastError();
}
cudaError_t launch_synth(cp4d_ctx *c, const float4 *P, int mode, float sigma, const float *g, float *out) {
    ProfScope ps(c, CP4D_K_SYNTH);
    const Dims &d = c->d;
    const size_t sh = (size_t)d.npi * d.m * sizeof(float);
    CP4D_DISPATCH_Q(d.Q, (k_synth<QQ><<<d.nz * d.n0, 128, sh, c->stream>>>(P, mode, sigma, g, out, c->phi, c->fwang, d.nd, d.na, d.npi, d.n0, d.nd, 0)));
    c->launches++;
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------
// reductions and vector helpers (power iteration, dot test)
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_dot(const float *__restrict__ x, const float *__restrict__ y, uint64_t n,
                                             double *slot) {
    double acc = 0.0;
    const uint64_t n4 = n / 4, stride = (uint64_t)gridDim.x * blockDim.x;
    const float4 *X = reinterpret_cast<const float4 *>(x), *Y = reinterpret_cast<const float4 *>(y);
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
        const float4 a = ld4(X + i), b = ld4(Y + i);
        acc += (double)a.x * b.x + (double)a.y * b.y + (double)a.z * b.z + (double)a.w * b.w;
    }
    if (blockIdx.x == 0 && threadIdx.x < (n & 3)) acc += (double)x[n4 * 4 + threadIdx.x] * y[n4 * 4 + threadIdx.x];
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    __shared__ double part[8];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += part[w];
        atomicAdd(slot, s);
    }
}

cudaError_t launch_sumsq_dot(cp4d_ctx *c, const float *x, const float *y, uint64_t n, double *slot) {
    ProfScope ps(c, CP4D_K_REDUCE);
    cudaError_t e = cudaMemsetAsync(slot, 0, sizeof(double), c->stream);
    if (e != cudaSuccess) return e;
    uint64_t blocks = (n / 4 + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    if (blocks < 1) blocks = 1;
    k_dot<<<(unsigned)blocks, 256, 0, c->stream>>>(x, y, n, slot);
    c->launches += 2;
    return cudaGetLastError();
}

__device__ __forceinline__ uint64_t splitmix(uint64_t x) {
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}
__global__ void __launch_bounds__(256) k_fill_normal(float *x, uint64_t n, uint64_t seed) {
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const uint64_t h = splitmix(seed * 0xD1342543DE82EF95ull + i);
        const float u1 = ((uint32_t)(h >> 40) + 1.0f) * (1.0f / 16777217.0f);  // (0,1]
        const float u2 = (uint32_t)(h & 0xFFFFFFu) * (1.0f / 16777216.0f);
        x[i] = sqrtf(-2.0f * logf(u1)) * cospif(2.0f * u2);
    }
}
cudaError_t launch_fill_normal(cp4d_ctx *c, float *x, uint64_t n, uint64_t seed) {
    ProfScope ps(c, CP4D_K_MISC);
    uint64_t blocks = (n + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    k_fill_normal<<<(unsigned)blocks, 256, 0, c->stream>>>(x, n, seed);
    c->launches++;
    return cudaGetLastError();
}

__global__ void __launch_bounds__(256) k_scale_diff(float *x, const float *a, const float *b,
                                                    float s, uint64_t n4) {
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    float4 *X = reinterpret_cast<float4 *>(x);
    const float4 *A = reinterpret_cast<const float4 *>(a), *B = reinterpret_cast<const float4 *>(b);
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride) {
        float4 v = A[i];
        if (B) { const float4 w = B[i]; v = sub4(v, w); }
        X[i] = make_float4(v.x * s, v.y * s, v.z * s, v.w * s);
    }
}
cudaError_t launch_scale_diff(cp4d_ctx *c, float *x, const float *a, const float *b, float s, uint64_t n) {
    ProfScope ps(c, CP4D_K_MISC);
    uint64_t blocks = (n / 4 + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    k_scale_diff<<<(unsigned)blocks, 256, 0, c->stream>>>(x, a, b, s, n / 4);  // V is a multiple of 4
    c->launches++;
    return cudaGetLastError();
}

}  // namespace cp4d
