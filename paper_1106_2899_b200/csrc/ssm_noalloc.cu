// ssm_noalloc.cu -- ssm_group_stress_noalloc (include/ssm.h): the group stresses of ssm_group_stress_device, computed
// without touching any memory the caller did not pass as an input or an output.
//
// Why it exists.  ssm_group_stress_device keeps its intermediate integer sums ([groups][13] int64) in the staging area of
// the ctx's workspace.  That is scratch memory, and some users of a coupling loop cannot provide or tolerate it:
//   - a flow solver that calls this library from inside a framework which owns the whole GPU through its own memory
//     pool (a raw cudaMalloc there either fails or takes memory the pool believes it has), and which hands the plug-in
//     only the buffers of its inputs and outputs;
//   - a step of a latency-critical loop, where cudaMalloc / cudaFree would synchronise the whole device;
//   - a caller whose staging area is busy: ssm_step_from_host and ssm_get_state / ssm_set_state of another stream's
//     work use the same bytes.
// For them the sums live in ONE file-scope device array below, of a fixed, stated size (kNoAllocMaxGroups groups,
// 416 KiB).  It is part of the library's image: every GPU on which libssm.so has been loaded holds it until the process
// exits, whether this entry point is ever called or not.
//
// What follows from sharing one array:
//   - it still holds the previous call's sums, so every call first clears the part it will use;
//   - two calls whose GPU work overlaps (two ctxs on two streams of one device, two host threads) race on it and both
//     get wrong answers.  Calls on ONE stream are ordered and safe.  Calls on different GPUs do not share anything (each
//     device has its own copy of the array);
//   - the name `g_group_sums` means the device array only inside device code.  In host code it is a host-side handle;
//     a kernel given `g_group_sums` as a pointer argument would fault or, on a machine where the GPU can reach host
//     memory, quietly add into the wrong bytes.  The host therefore asks the runtime for the real device address
//     (cudaGetSymbolAddress), once per device and with that device current, and passes that to the kernels.
// The first call on a device does that look-up (it may also make the runtime load this module's code onto the device),
// so make that first call before starting any stream capture.
//
// No cudaMalloc, cudaFree, cudaMallocAsync or other allocating routine is called here; the clear is a cudaMemsetAsync
// on the ctx's stream.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/ssm.h"
#include "ssm_common.h"

namespace ssm {
void ctx_view(const ssm_ctx *c, CtxView *v);
int ctx_fail(ssm_ctx *c, int code, const char *msg);
void ctx_add_launches(ssm_ctx *c, int n);
}  // namespace ssm

using namespace ssm;

namespace {

constexpr long long kNoAllocMaxGroups = SSM_NOALLOC_MAX_GROUPS;     // 4096 groups x 13 sums x 8 B = 425,984 B
constexpr int kMaxDevices = 64;

// The scratch: fixed-point sums [group][13] (sigma[6], sigma_v[6], Z), 2^-kStressShift.  Device copy per GPU.
static __device__ __align__(256) long long g_group_sums[kNoAllocMaxGroups * 13];

// Device address of g_group_sums on each GPU, looked up on first use (null = not yet).
std::mutex g_setup_mutex;
long long *g_sums_addr[kMaxDevices] = {};

// Variant of ssm_group_stress_kernel (ssm_aux.cu) with the same arithmetic in the same order -- per-chain sigma (eq 16)
// and sigma^(v) (eq 76) in fp32, rounded once to 2^-kStressShift, then integer sums -- so that its results equal that
// kernel's bit for bit whatever the order of the atomics.  One thread per chain; `sums` is the device address of
// g_group_sums, cleared by the caller for the groups in use.
__global__ void __launch_bounds__(128) ssm_group_stress_noalloc_kernel(const unsigned char *state, long long *sums, int N,
                                                                       long long M, long long cpg, float cs)
{
    const long long k0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = k0 < M;
    const long long k = valid ? k0 : M - 1;
    const int NP = padded_beads(N);
    float sg[6] = {0, 0, 0, 0, 0, 0}, sv[6] = {0, 0, 0, 0, 0, 0};
    float p[3], q[3];
    for (int c = 0; c < 3; ++c) p[c] = *reinterpret_cast<const float *>(state + off_R(k, NP, 0, c));
    for (int i = 1; i < N; ++i) {
        float b[3];
        for (int c = 0; c < 3; ++c) { q[c] = *reinterpret_cast<const float *>(state + off_R(k, NP, i, c)); b[c] = q[c] - p[c]; p[c] = q[c]; }
        sg[0] += fmaf(3.f * b[0], b[0], -1.f); sg[1] += fmaf(3.f * b[1], b[1], -1.f); sg[2] += fmaf(3.f * b[2], b[2], -1.f);
        sg[3] = fmaf(3.f * b[0], b[1], sg[3]); sg[4] = fmaf(3.f * b[1], b[2], sg[4]); sg[5] = fmaf(3.f * b[2], b[0], sg[5]);
    }
    sg[0] -= 1.f; sg[1] -= 1.f; sg[2] -= 1.f;                 // 3 sum b^2 - N = sum (3 b^2 - 1) - 1
    const int Z = *reinterpret_cast<const int *>(state + off_Z(k, NP));
    for (int j = 0; j < Z; ++j) {
        const int s = state[off_S(k, NP, j)] - 1;
        float d[3];
        for (int c = 0; c < 3; ++c)
            d[c] = *reinterpret_cast<const float *>(state + off_R(k, NP, s, c)) - *reinterpret_cast<const float *>(state + off_A(k, NP, j, c));
        sv[0] += fmaf(cs * d[0], d[0], -1.f); sv[1] += fmaf(cs * d[1], d[1], -1.f); sv[2] += fmaf(cs * d[2], d[2], -1.f);
        sv[3] = fmaf(cs * d[0], d[1], sv[3]); sv[4] = fmaf(cs * d[1], d[2], sv[4]); sv[5] = fmaf(cs * d[2], d[0], sv[5]);
    }
    const long long group = k / cpg;
    const bool one_group = __all_sync(0xffffffffu, group == __shfl_sync(0xffffffffu, group, 0));
    constexpr float scale = (float)(1 << kStressShift);
    for (int t = 0; t < 13; ++t) {
        long long v = t < 6 ? __float2ll_rn(sg[t] * scale) : (t < 12 ? __float2ll_rn(sv[t - 6] * scale) : (long long)Z << kStressShift);
        if (!valid) v = 0;
        if (one_group) {        // the usual case: a warp's 32 chains sit in one group -> one atomic per warp and component
            for (int o = 16; o >= 1; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
            if ((threadIdx.x & 31) == 0) atomicAdd(reinterpret_cast<unsigned long long *>(sums + group * 13 + t), (unsigned long long)v);
        } else if (valid) atomicAdd(reinterpret_cast<unsigned long long *>(sums + group * 13 + t), (unsigned long long)v);
    }
}

// out[g][t] = sums[g][t] / (2^kStressShift * chains in group g): the means of eq 54 over each group.
__global__ void __launch_bounds__(256) ssm_group_mean_noalloc_kernel(const long long *sums, double *out, long long n_groups,
                                                                     long long M, long long cpg)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_groups * 13) return;
    const long long g = i / 13, n = (g + 1) * cpg <= M ? cpg : M - g * cpg;
    out[i] = (double)sums[i] / ((double)(1 << kStressShift) * (double)n);
}

// Device address of g_group_sums on the CURRENT device `dev` (set-up on first use, under a lock).
cudaError_t scratch_address(int dev, long long **ptr)
{
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_sums_addr[dev]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_group_sums);
        if (e != cudaSuccess) return e;
        g_sums_addr[dev] = static_cast<long long *>(p);
    }
    *ptr = g_sums_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int ssm_group_stress_noalloc(ssm_ctx *c, int64_t chains_per_group, double *d_out)
{
    if (!c) return ctx_fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!d_out) return ctx_fail(c, SSM_EINVAL, "d_out is NULL");
    if (chains_per_group < 1) return ctx_fail(c, SSM_EINVAL, "chains_per_group must be >= 1");
    CtxView v;
    ctx_view(c, &v);
    const long long M = v.n_chains, cpg = chains_per_group < M ? chains_per_group : M, ng = (M + cpg - 1) / cpg;
    if (ng > kNoAllocMaxGroups)
        return ctx_fail(c, SSM_ERANGE, "ssm_group_stress_noalloc: more than SSM_NOALLOC_MAX_GROUPS (4096) groups; the built-in "
                                       "scratch array is fixed at that size -- use larger groups or ssm_group_stress_device");
    // The array's address belongs to one device: the GPU that holds the ctx's state must be the current one.
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return ctx_fail(c, SSM_ECUDA, cudaGetErrorString(e));
    cudaPointerAttributes attr;
    e = cudaPointerGetAttributes(&attr, v.state);
    if (e != cudaSuccess) return ctx_fail(c, SSM_ECUDA, cudaGetErrorString(e));
    if (attr.type != cudaMemoryTypeDevice || attr.device != dev)
        return ctx_fail(c, SSM_EINVAL, "ssm_group_stress_noalloc: the GPU that holds the ctx's workspace must be the current device");
    if (dev < 0 || dev >= kMaxDevices) return ctx_fail(c, SSM_EINVAL, "ssm_group_stress_noalloc: device ordinal beyond 63");
    long long *sums = nullptr;
    e = scratch_address(dev, &sums);
    if (e != cudaSuccess) return ctx_fail(c, SSM_ECUDA, cudaGetErrorString(e));

    cudaStream_t st = static_cast<cudaStream_t>(v.stream);
    // the array keeps the last call's sums: clear the groups this call adds into
    e = cudaMemsetAsync(sums, 0, (size_t)ng * 13 * sizeof(long long), st);
    if (e != cudaSuccess) return ctx_fail(c, SSM_ECUDA, cudaGetErrorString(e));
    ssm_group_stress_noalloc_kernel<<<(unsigned)((M + 127) / 128), 128, 0, st>>>(v.state, sums, v.n_beads, M, cpg, v.cs);
    e = cudaGetLastError();
    if (e != cudaSuccess) return ctx_fail(c, SSM_ECUDA, cudaGetErrorString(e));
    ssm_group_mean_noalloc_kernel<<<(unsigned)((ng * 13 + 255) / 256), 256, 0, st>>>(sums, d_out, ng, M, cpg);
    e = cudaGetLastError();
    if (e != cudaSuccess) return ctx_fail(c, SSM_ECUDA, cudaGetErrorString(e));
    ctx_add_launches(c, 2);
    return SSM_OK;
}
