// cp4d_forward_static: the forward operator g = K1 f (Eq. 9; pi-fold L198-L202) for callers that cannot hand the
// library a place for its scratch at call time -- code under CUDA graph capture, serving loops, harnesses that forbid device
// allocation.  The forward projector's only scratch, the partial ray sums P[z][i][b][j] (m * n_theta0 * nd * nz floats), lives
// here in a file-scope __device__ array of CP4D_STATIC_SCRATCH_BYTES instead of in the workspace region cp4d_forward uses; the
// kernels are the same ones (launch_forward_partial + launch_synth), so the result is the one of cp4d_forward up to the order
// of the projector's RED additions.
//
// The array is held by every GPU that loads the library until the process exits.  In HOST code the array's name is a host-side
// stand-in, not a device address: the address the kernels get comes from cudaGetSymbolAddress, asked once per device with that
// device current (static_psum below).  All calls on one device share the array and it keeps the last call's contents: every
// call zero-fills the part it uses (launch_forward_partial does, on the context's stream), and two calls that overlap on the
// GPU (different streams, no dependency) race on it.
#include <cstdio>
#include <mutex>

#include "cp4d_internal.cuh"

namespace cp4d {

namespace {

static_assert(CP4D_STATIC_SCRATCH_BYTES % 256 == 0, "whole 256-byte units");
static __device__ __align__(256) float4 g_psum_static[CP4D_STATIC_SCRATCH_BYTES / sizeof(float4)];

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
float4 *g_psum_addr[MAX_DEVICES] = {};      // device address of g_psum_static on each device, asked once

// the context's device is current (the entry point's guard): device address of the array on this device
cudaError_t static_psum(int device, float4 **out) {
    if (device < 0 || device >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_psum_addr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_psum_static);
        if (e != cudaSuccess) return e;
        g_psum_addr[device] = static_cast<float4 *>(p);
    }
    *out = g_psum_addr[device];
    return cudaSuccess;
}

struct DeviceScope {      // makes the context's device current for the call and puts the caller's back
    int prev = -1;
    explicit DeviceScope(int dev) {
        int cur = -1;
        if (cudaGetDevice(&cur) != cudaSuccess) { cudaGetLastError(); cur = -1; }
        if (cur != dev && cudaSetDevice(dev) == cudaSuccess) prev = cur;
    }
    ~DeviceScope() {
        if (prev >= 0) cudaSetDevice(prev);
    }
    DeviceScope(const DeviceScope &) = delete;
    DeviceScope &operator=(const DeviceScope &) = delete;
};

int fail_static(cp4d_ctx *c, int code, const char *what, cudaError_t e = cudaSuccess) {
    c->err = what;
    if (e != cudaSuccess) { c->err += ": "; c->err += cudaGetErrorString(e); cudaGetLastError(); }
    return code;
}

bool ranges_overlap(const void *a, uint64_t na, const void *b, uint64_t nb) {
    const uintptr_t a0 = (uintptr_t)a, b0 = (uintptr_t)b;
    return a0 < b0 + nb && b0 < a0 + na;
}

}  // namespace

}  // namespace cp4d

using namespace cp4d;

extern "C" int cp4d_forward_static(cp4d_ctx *ctx, const float *f, float *g) {
    if (!ctx) return CP4D_EINVAL;
    DeviceScope scope(ctx->device);
    const Dims &d = ctx->d;
    if (!f || !g || ((uintptr_t)f & 15) || ((uintptr_t)g & 15) || ranges_overlap(f, d.V * 4, g, d.S * 4))
        return fail_static(ctx, CP4D_EINVAL, "forward_static: bad pointers");
    const uint64_t need = (uint64_t)d.nz * d.n0 * d.nd * d.m * sizeof(float);
    if (need > (uint64_t)CP4D_STATIC_SCRATCH_BYTES) {
        char msg[200];
        std::snprintf(msg, sizeof msg, "forward_static: the partial ray sums of this problem need %llu bytes, the static scratch array holds %llu (CP4D_STATIC_SCRATCH_BYTES); use cp4d_forward",
                      (unsigned long long)need, (unsigned long long)CP4D_STATIC_SCRATCH_BYTES);
        return fail_static(ctx, CP4D_ETOOLARGE, msg);
    }
    float4 *P = nullptr;
    cudaError_t e = static_psum(ctx->device, &P);
    if (e != cudaSuccess) return fail_static(ctx, CP4D_ECUDA, "forward_static: cudaGetSymbolAddress", e);
    if (d.nf) {      // frame mode with N_t > M: K1 includes the analysis f_j = sum_q phi_j(t_q) f(t_q), as in cp4d_forward
        if ((e = launch_mix(ctx, f, ctx->cf, d.m, d.nf, d.nf, 1)) != cudaSuccess) return fail_static(ctx, CP4D_ECUDA, "forward_static: analysis", e);
        f = ctx->cf;
    }
    // zero-fills the used part of P on the context's stream, then the projector REDs its partial ray sums into it
    if ((e = launch_forward_partial(ctx, f, P)) != cudaSuccess) return fail_static(ctx, CP4D_ECUDA, "forward_static: forward_partial", e);
    if ((e = launch_synth(ctx, P, 0, 0.f, nullptr, g)) != cudaSuccess) return fail_static(ctx, CP4D_ECUDA, "forward_static: synth", e);
    return CP4D_OK;
}
