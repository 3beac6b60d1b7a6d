// ssm_api.cu -- the C ABI of libssm.so (include/ssm.h): argument checking, workspace
// carve-up, host-side tables and launch sequencing.  Every step of the method runs in the
// kernels of ssm_step.cu / ssm_aux.cu; nothing here computes on chains.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/ssm.h"
#include "ssm_common.h"
#include "ssm_rng.cuh"

namespace ssm {
cudaError_t step_occupancy(int n_beads, int *blocks_per_sm);
cudaError_t launch_step(int n_beads, const StepParams &p, int grid, cudaStream_t st);
cudaError_t launch_init(const InitParams &p, cudaStream_t st);
cudaError_t measure_rates(unsigned *d_scratch, int blocks, cudaStream_t st, double cycles[8]);
cudaError_t launch_xfer(bool do_export, unsigned char *state, float *R, float *A, unsigned char *S, int N,
                        long long k0, long long nk, long long pitch, int hide_low, int *bad_state, cudaStream_t st);
cudaError_t launch_clear_low(unsigned char *state, long long n_tiles, cudaStream_t st);
cudaError_t launch_group_stress(const unsigned char *state, long long *out, int N, long long M, long long cpg, float cs,
                                cudaStream_t st);
cudaError_t launch_recenter(unsigned char *state, int N, long long M, cudaStream_t st);
cudaError_t launch_kappa(const double *d_kappa, float *out, long long n, double dt, cudaStream_t st);
cudaError_t launch_group_mean(const long long *sums, double *out, long long n_groups, long long M, long long cpg,
                              cudaStream_t st);
cudaError_t launch_chain_stress(const unsigned char *state, float *out, int N, long long M, float cs, cudaStream_t st);
cudaError_t launch_corr(const CorrParams &c, cudaStream_t st);
cudaError_t launch_bm_calib(float bm0, int n_cand, double *d_out, cudaStream_t st);
}  // namespace ssm

using namespace ssm;

static thread_local std::string g_err;   // errors without a ctx

struct Layout {
    size_t state, stress, kappa, counter, samples, ring, accf, accg, csum, stage, total;
    long long n_tiles, stage_chains;
};

struct ssm_ctx {
    ssm_params p;
    Layout lay;
    unsigned char *ws;
    cudaStream_t st;
    long long step;          // global step counter
    long long n_records;     // stress samples recorded since the last reset
    int fuse, grid, grid_default;
    long long launches;
    bool springs_on;
    int low_mode;            // encoding of the anchors' fourth word: 0 all zero, 1 fp32 low part of x (simple shear),
                             // 2 three packed 10-bit low parts (general tensor)
    StepParams sp;           // constant part filled at init
    // correlator schedule (identical for all chains) and product counts, host side
    unsigned char cpos[kCorrMaxLevels], cfil[kCorrMaxLevels], cpar[kCorrMaxLevels];
    std::vector<long long> ccount;      // [L][P] insertions with a product at (level, bin)
    std::vector<float> kappa_host;      // dt kappa of the last ssm_step_kappa call, [groups][9]
    bool state_valid = true;            // false after an import that failed half way (CUDA error): stepping is refused until a state is imported again
    double calib[8] = {0, 0, 0, 0, 0, 0, 0, 0};   // ssm_noise_calibration: the record of calibrate_bm for bm_noise
    cudaStream_t copy_st = nullptr;     // ssm_step_from_host: uploads run here, beside the stepping on st
    cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
    std::string err;
};

static int fail(ssm_ctx *c, int code, const std::string &msg)
{
    if (c) c->err = msg; else g_err = msg;
    return code;
}
static int cuda_fail(ssm_ctx *c, cudaError_t e, const char *what)
{
    return fail(c, SSM_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CK(c, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail((c), e_, #call); } while (0)

constexpr int kCalibCand = 9;      // neighbouring floats tried around the first estimate of a Box-Muller constant

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

static bool check_params(const ssm_params *p, std::string &why)
{
    if (!p) { why = "params is NULL"; return false; }
    const int N = p->n_beads;
    if (N < 2 || N > 128) { why = "n_beads must be 2..128"; return false; }
    if (p->n_chains < 1) { why = "n_chains must be >= 1"; return false; }
    if (p->chain_offset + (uint64_t)p->n_chains + 16 > 0xFFFFFFFFull) { why = "global chain index must fit 32 bits"; return false; }
    if (!(p->dt > 0.0) || !(p->dt < 1.0 / 6.0)) { why = "dt must be in (0, 1/6): the Euler map needs 12 dt < 2"; return false; }
    if (!(p->n_s > 0.0)) { why = "n_s must be > 0"; return false; }
    if (!(p->zeta_s > 0.0)) { why = "zeta_s must be > 0"; return false; }
    if (p->k_attempts < 0) { why = "k_attempts must be >= 0"; return false; }
    if (p->stage_chains < 0) { why = "stage_chains must be >= 0"; return false; }
    if (p->stress_every < 0 || p->sample_every < 0 || p->stress_capacity < 0) { why = "negative sampling parameter"; return false; }
    if (p->stress_every > 0 && p->stress_capacity < 1) { why = "stress_capacity must be >= 1 when stress_every > 0"; return false; }
    if (p->sample_every > 0) {
        if (p->corr_levels < 1 || p->corr_levels > kCorrMaxLevels) { why = "corr_levels must be 1..32"; return false; }
        if (p->corr_bins < 2 || p->corr_bins > 32 || (p->corr_bins & 1)) { why = "corr_bins must be even, 2..32"; return false; }
        if (p->corr_groups < 1 || p->corr_groups > 1024) { why = "corr_groups must be 1..1024"; return false; }
        if (!(p->corr_components == 0 || p->corr_components == 1 || p->corr_components == 3)) { why = "corr_components must be 0, 1 or 3"; return false; }
    }
    return true;
}

static Layout make_layout(const ssm_params *p)
{
    Layout L{};
    const int npad = padded_beads(p->n_beads), cpw = chains_per_warp(npad);
    L.n_tiles = (p->n_chains + cpw - 1) / cpw;
    size_t o = 0;
    L.state = o; o = align_up(o + (size_t)L.n_tiles * kTileBytes, 256);
    L.stress = o; o = align_up(o + (size_t)p->stress_capacity * 12 * 8, 256);
    L.kappa = o; o = align_up(o + (size_t)L.n_tiles * 9 * 4, 256);        // dt kappa per group (at most one group per tile)
    L.counter = o; o = align_up(o + 3 * sizeof(int), 256);                 // tile counters of the step kernel [0], [1]; [2] = "the imported state was malformed"
    const bool corr = p->sample_every > 0;
    const size_t M = (size_t)p->n_chains;
    const size_t Mv = M * (size_t)(p->corr_components == 3 ? 3 : 1);      // histories: one per chain and component
    L.samples = o; if (corr) o = align_up(o + (size_t)kMaxFuse * Mv * 8, 256);
    L.ring = o; if (corr) o = align_up(o + (size_t)p->corr_levels * p->corr_bins * Mv * 4, 256);
    L.accf = o; if (corr) o = align_up(o + (size_t)p->corr_levels * Mv * 4, 256);
    L.accg = o; if (corr) o = align_up(o + (size_t)p->corr_levels * Mv * 4, 256);
    // two sum arrays: f_new g_old (eq 43) and g_new g_old (eq 66)
    L.csum = o; if (corr) o = align_up(o + 2 * (size_t)p->corr_groups * p->corr_levels * p->corr_bins * 8, 256);
    // staging for host-pointer get/set state and chain stress: chunks of <= 65536 chains
    const long long want_stage = p->stage_chains > 0 ? p->stage_chains : 65536;
    L.stage_chains = p->n_chains < want_stage ? p->n_chains : want_stage;
    // (at least 1 MB, so that the issue-rate probe's scratch of 2 kB per SM fits any ensemble)
    size_t stage_bytes = (size_t)L.stage_chains * (size_t)(29 * npad > 48 ? 29 * npad : 48);
    if (stage_bytes < ((size_t)1 << 20)) stage_bytes = (size_t)1 << 20;
    L.stage = o; o = align_up(o + stage_bytes, 256);
    L.total = o;
    return L;
}

// "u < p" with u = (k + 1/2) 2^-23  <=>  k < T(p) = ceil(p 2^23 - 1/2)
static unsigned threshold23(double p)
{
    double t = std::ceil(p * 8388608.0 - 0.5);
    if (t < 0.0) t = 0.0;
    if (t > 8388608.0) t = 8388608.0;
    return (unsigned)t;
}

extern "C" size_t ssm_workspace_bytes(const ssm_params *p)
{
    std::string why;
    if (!check_params(p, why)) { g_err = why; return 0; }
    return make_layout(p).total;
}

static void corr_clear(ssm_ctx *c)
{
    std::memset(c->cpos, 0, sizeof c->cpos); std::memset(c->cfil, 0, sizeof c->cfil); std::memset(c->cpar, 0, sizeof c->cpar);
    c->ccount.assign((size_t)kCorrMaxLevels * 32, 0);
}

static int clear_accumulators(ssm_ctx *c)
{
    const ssm_params &p = c->p;
    if (p.stress_capacity > 0)
        CK(c, cudaMemsetAsync(c->ws + c->lay.stress, 0, (size_t)p.stress_capacity * 12 * 8, c->st));
    if (p.sample_every > 0) {
        CK(c, cudaMemsetAsync(c->ws + c->lay.ring, 0, c->lay.stage - c->lay.ring, c->st));
        corr_clear(c);
    }
    c->n_records = 0;
    return SSM_OK;
}

// ---------------------------------------------------------------------------------------
// Calibrated Box-Muller constant.  The kernels draw N(0, sigma2) as r cos, r sin with
// r^2 = bm log2(u_a), bm = -2 ln2 sigma2 in fp32, on 2^16 radius codes and 2^16 angle codes through the special-function
// unit.  The variance that comes out is a finite sum, which ssm_bm_calib_kernel forms for a constant and its neighbouring
// floats; here the float is chosen whose variance is nearest the exact one of the discrete law,
//   sigma2 * mean_ka(-2 ln u_a) * 1/2        (the mean of cos^2 over the uniform angle grid is exactly 1/2),
// which removes the fp32 rounding of bm and the (non-zero-mean) error of lg2 / sqrt / sin / cos from the amplitude, down
// to half an ulp of bm (<= 3.4e-8 of the variance).  Costs no instruction in the kernels.  Two tiny launches and one
// synchronisation of the stream, once per (device, sigma2) in the process: the result is cached.
// rec (may be null) [8]: nominal bm, calibrated bm, relative variance error at the nominal and at the calibrated
// constant, mean cos^2 - 1/2, mean sin^2 - 1/2, ulps moved, 0.
// ---------------------------------------------------------------------------------------
struct CalibEntry { float bm; double rec[8]; };
static std::mutex g_calib_mutex;
static std::map<std::pair<int, unsigned>, CalibEntry> g_calib_cache;

static double exact_mean_r2()        // mean over the 2^16 codes of -2 ln u_a, u_a = (ka + 1/2) 2^-16
{
    static const double v = [] { double s = 0.0; for (int k = 65535; k >= 0; --k) s += -2.0 * std::log(((double)k + 0.5) / 65536.0); return s / 65536.0; }();
    return v;
}

static cudaError_t calibrate_bm(int dev, double sigma2, double *d_scratch, cudaStream_t st, float *bm_out, double *rec)
{
    const float nominal = (float)(-2.0 * 0.6931471805599453 * sigma2);
    unsigned bits; std::memcpy(&bits, &nominal, 4);
    std::lock_guard<std::mutex> lock(g_calib_mutex);
    auto it = g_calib_cache.find({dev, bits});
    if (it == g_calib_cache.end()) {
        const double target = sigma2 * exact_mean_r2() * 0.5;
        double h[kCalibCand + 2] = {};
        auto variance = [&](int c, int n) { return (h[c] / 65536.0) * (0.5 * (h[n] + h[n + 1]) / 65536.0); };
        cudaError_t e;
        if ((e = launch_bm_calib(nominal, 1, d_scratch, st)) != cudaSuccess
            || (e = cudaMemcpyAsync(h, d_scratch, 3 * sizeof(double), cudaMemcpyDeviceToHost, st)) != cudaSuccess
            || (e = cudaStreamSynchronize(st)) != cudaSuccess) return e;
        CalibEntry en{};
        en.rec[0] = nominal;
        en.rec[2] = variance(0, 1) / target - 1.0;
        en.rec[4] = h[1] / 65536.0 - 0.5; en.rec[5] = h[2] / 65536.0 - 0.5;
        const float centre = (float)((double)nominal * target / variance(0, 1));
        if ((e = launch_bm_calib(centre, kCalibCand, d_scratch, st)) != cudaSuccess
            || (e = cudaMemcpyAsync(h, d_scratch, (kCalibCand + 2) * sizeof(double), cudaMemcpyDeviceToHost, st)) != cudaSuccess
            || (e = cudaStreamSynchronize(st)) != cudaSuccess) return e;
        int best = kCalibCand / 2;
        for (int cnd = 0; cnd < kCalibCand; ++cnd)
            if (std::fabs(variance(cnd, kCalibCand) - target) < std::fabs(variance(best, kCalibCand) - target)) best = cnd;
        int cb; std::memcpy(&cb, &centre, 4);
        cb += best - kCalibCand / 2;
        std::memcpy(&en.bm, &cb, 4);
        en.rec[1] = en.bm;
        en.rec[3] = variance(best, kCalibCand) / target - 1.0;
        int nb; std::memcpy(&nb, &nominal, 4);
        en.rec[6] = (double)(cb - nb);
        it = g_calib_cache.emplace(std::make_pair(dev, bits), en).first;
    }
    *bm_out = it->second.bm;
    if (rec) std::memcpy(rec, it->second.rec, sizeof it->second.rec);
    return cudaSuccess;
}

extern "C" int ssm_init(ssm_ctx **out, const ssm_params *p, void *d_workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!out) return fail(nullptr, SSM_EINVAL, "out is NULL");
    *out = nullptr;
    std::string why;
    if (!check_params(p, why)) return fail(nullptr, SSM_EINVAL, why);
    const Layout lay = make_layout(p);
    if (!d_workspace || workspace_bytes < lay.total) return fail(nullptr, SSM_ENOMEM, "workspace too small");
    if (((uintptr_t)d_workspace & 255u) != 0) return fail(nullptr, SSM_ENOMEM, "workspace must be 256-byte aligned");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) return fail(nullptr, SSM_ECUDA, "no CUDA device (there is no CPU fallback)");

    ssm_ctx *c = new (std::nothrow) ssm_ctx();
    if (!c) return fail(nullptr, SSM_ENOMEM, "host allocation failed");
    c->p = *p; c->lay = lay; c->ws = (unsigned char *)d_workspace; c->st = (cudaStream_t)cuda_stream;
    c->step = 0; c->n_records = 0; c->fuse = kMaxFuse; c->launches = 0; c->low_mode = 0;
    c->springs_on = p->n_0 > 0.0 && std::isfinite(p->n_0);
    corr_clear(c);

    int dev = 0, n_sm = 0, bps = 0;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess || (e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess
        || (e = step_occupancy(padded_beads(p->n_beads), &bps)) != cudaSuccess) {
        int rc = cuda_fail(nullptr, e, "device query"); delete c; return rc;
    }
    if (bps < 1) { delete c; return fail(nullptr, SSM_ECUDA, "step kernel does not fit on an SM"); }
    const long long want = (lay.n_tiles + kWarpsPerBlock - 1) / kWarpsPerBlock;
    const long long cap = (long long)n_sm * bps;
    c->grid = c->grid_default = (int)(want < cap ? want : cap);

    // constant launch parameters and integer decision thresholds (fp64 on the host)
    const double h = p->dt / p->zeta_s;
    StepParams &sp = c->sp;
    std::memset(&sp, 0, sizeof sp);
    sp.state = c->ws + lay.state;
    sp.n_chains = p->n_chains; sp.chain_offset = p->chain_offset; sp.n_tiles = (int)lay.n_tiles;
    philox_round_keys((unsigned)(p->seed & 0xFFFFFFFFull), (unsigned)(p->seed >> 32), sp.rk);
    sp.springs_on = c->springs_on ? 1 : 0;
    sp.k_attempts = p->k_attempts;
    sp.n_act = p->n_beads;
    sp.n_comp = p->corr_components == 3 ? 3 : 1;
    sp.dt3 = (float)(3.0 * p->dt);
    // the three Box-Muller constants, each calibrated on this device (calibrate_bm above; cached per process)
    float bm_bond = 0.0f;
    {
        double *d_cal = reinterpret_cast<double *>(c->ws + lay.stage);
        if ((e = calibrate_bm(dev, 2.0 * p->dt, d_cal, c->st, &sp.bm_noise, c->calib)) != cudaSuccess             // eqs 44, 46, 47
            || (e = calibrate_bm(dev, p->n_s / 3.0, d_cal, c->st, &sp.bm_anchor, nullptr)) != cudaSuccess        // eqs 15, 52
            || (e = calibrate_bm(dev, 1.0 / 3.0, d_cal, c->st, &bm_bond, nullptr)) != cudaSuccess) {             // eq 6
            int rc = cuda_fail(nullptr, e, "Box-Muller calibration"); delete c; return rc;
        }
    }
    sp.fx_scale = (float)(p->dt * (3.0 / p->n_s) * (double)(1 << kFxShift));
    sp.q2l = (float)(2.0 * (3.0 / (4.0 * p->n_s)) * 1.4426950408889634);
    sp.h2 = (float)(2.0 * h);
    sp.cs = (float)(3.0 / p->n_s);
    sp.t_destroy = threshold23(std::fmin(h, 1.0));
    for (int K = 1; K <= 128; ++K) {
        const double pc = c->springs_on ? std::fmin(h / (p->n_0 * (double)K), 0.5) : 0.0;
        sp.t_c1[K] = threshold23(pc); sp.t_c2[K] = threshold23(2.0 * pc);
        sp.h_c2[K] = sp.t_c2[K] ? (int)((sp.t_c2[K] - 1u) >> 7) : -1;
    }

    InitParams ip;
    std::memset(&ip, 0, sizeof ip);
    ip.state = c->ws + lay.state;
    ip.n_chains_padded = lay.n_tiles * chains_per_warp(padded_beads(p->n_beads)); ip.n_chains = p->n_chains;
    ip.n_pad = padded_beads(p->n_beads);
    ip.chain_offset = p->chain_offset; std::memcpy(ip.rk, sp.rk, sizeof ip.rk);
    ip.n_beads = p->n_beads; ip.springs_on = sp.springs_on;
    ip.bm_bond = bm_bond; ip.bm_anchor = sp.bm_anchor;
    if (c->springs_on) {       // Poisson(N/N0) CDF (eq 12) as integer thresholds
        const double lam = (double)p->n_beads / p->n_0;
        double pmf = std::exp(-lam), cdf = 0.0;
        for (int z = 0; z < p->n_beads; ++z) {
            if (z > 0) pmf = pmf * lam / (double)z;
            cdf += pmf;
            ip.t_cdf[z] = threshold23(cdf);
        }
    }
    sp.tile_counter = reinterpret_cast<int *>(c->ws + lay.counter); sp.counter_slot = 0;
    if ((e = cudaMemsetAsync(c->ws + lay.counter, 0, 3 * sizeof(int), c->st)) != cudaSuccess
        || (e = cudaMemsetAsync(c->ws + lay.state, 0, (size_t)lay.n_tiles * kTileBytes, c->st)) != cudaSuccess
        || (e = launch_init(ip, c->st)) != cudaSuccess) {
        int rc = cuda_fail(nullptr, e, "ssm_init launch"); delete c; return rc;
    }
    c->launches += 1;
    int rc = clear_accumulators(c);
    if (rc != SSM_OK) { g_err = c->err; delete c; return rc; }
    *out = c;
    return SSM_OK;
}

// advance the host copy of the correlator schedule by one sample, counting products
static void corr_schedule_sample(ssm_ctx *c)
{
    const int L = c->p.corr_levels, Pb = c->p.corr_bins;
    for (int lev = 0; lev < L; ++lev) {
        if (c->cfil[lev] < Pb) ++c->cfil[lev];
        const int kmin = lev == 0 ? 0 : Pb / 2;
        for (int q = kmin; q < c->cfil[lev]; ++q) c->ccount[(size_t)lev * 32 + q] += 1;
        c->cpos[lev] = (unsigned char)((c->cpos[lev] + 1) % Pb);
        if (c->cpar[lev] == 0) { c->cpar[lev] = 1; break; }
        c->cpar[lev] = 0;
    }
}

// the launch parameters of the next T <= fuse steps (records and samples due, where they go); the caller adds the flow
static StepParams block_params(ssm_ctx *c, long long step, long long n_records, int T, long long *nrec_out, long long *nsmp_out)
{
    const ssm_params &p = c->p;
    StepParams sp = c->sp;
    sp.step0 = (unsigned long long)step; sp.n_fuse = T;
    long long nrec = 0, nsmp = 0;
    if (p.stress_every > 0) nrec = (step + T) / p.stress_every - step / p.stress_every;
    if (p.sample_every > 0) nsmp = (step + T) / p.sample_every - step / p.sample_every;
    sp.rec_mask = 0u; sp.smp_mask = 0u;
    for (int n = 0; n < T; ++n) {
        if (p.stress_every > 0 && (step + n + 1) % p.stress_every == 0) sp.rec_mask |= 1u << n;
        if (p.sample_every > 0 && (step + n + 1) % p.sample_every == 0) sp.smp_mask |= 1u << n;
    }
    sp.n_rec = (int)nrec;
    sp.stress = reinterpret_cast<long long *>(c->ws + c->lay.stress) + n_records * 12;
    sp.samples = nsmp > 0 ? reinterpret_cast<float2 *>(c->ws + c->lay.samples) : nullptr;
    *nrec_out = nrec; *nsmp_out = nsmp;
    return sp;
}

// steps of the next launch: at most the fusion depth, and never across a multiple of 2^32 steps (the kernel forms the
// part of its Philox calls that depends on the step's high bits once per tile: ssm_rng.cuh, stream_prefix)
static int next_block(const ssm_ctx *c, long long step, long long left)
{
    long long T = left < c->fuse ? left : c->fuse;
    const long long to_wrap = 0x100000000ll - (step & 0xFFFFFFFFll);
    return (int)(T < to_wrap ? T : to_wrap);
}

// advance n_steps under simple shear (d_kappa null) or under the device table of tensors d_kappa
static int step_impl(ssm_ctx *c, int64_t n_steps, double shear_rate, const float *d_kappa, long long tiles_per_group)
{
    const ssm_params &p = c->p;
    if (!c->state_valid) return fail(c, SSM_ESTATE, "a state import failed half way: import a state again before stepping");
    if (p.stress_every > 0) {
        const long long need = (c->step + n_steps) / p.stress_every - c->step / p.stress_every;
        if (c->n_records + need > p.stress_capacity) return fail(c, SSM_ERANGE, "stress buffer would overflow (stress_capacity)");
    }
    const float gdt = d_kappa ? 0.0f : (float)(shear_rate * p.dt);
    // the fourth word of an anchor is the low part of its compensated advection; simple shear and the
    // general tensor encode it differently, so it restarts from zero when the kind of flow changes
    const int want = d_kappa ? 2 : (gdt != 0.0f ? 1 : 0);
    if (n_steps > 0 && want != 0 && c->springs_on) {
        if (c->low_mode != 0 && c->low_mode != want) {
            CK(c, launch_clear_low(c->ws + c->lay.state, c->lay.n_tiles, c->st));
            c->launches += 1;
        }
        c->low_mode = want;
    }
    long long left = n_steps;
    while (left > 0) {
        const int T = next_block(c, c->step, left);
        long long nrec = 0, nsmp = 0;
        StepParams sp = block_params(c, c->step, c->n_records, T, &nrec, &nsmp);
        sp.gdt = gdt; sp.kappa = d_kappa; sp.tiles_per_group = (int)tiles_per_group;
        sp.counter_slot = c->sp.counter_slot;
        CK(c, launch_step(padded_beads(p.n_beads), sp, c->grid, c->st));
        c->sp.counter_slot ^= 1;
        c->launches += 1;
        if (nsmp > 0) {
            CorrParams cp;
            std::memset(&cp, 0, sizeof cp);
            cp.samples = sp.samples;
            cp.ring = reinterpret_cast<float *>(c->ws + c->lay.ring);
            cp.acc_f = reinterpret_cast<float *>(c->ws + c->lay.accf);
            cp.acc_g = reinterpret_cast<float *>(c->ws + c->lay.accg);
            cp.sum = reinterpret_cast<long long *>(c->ws + c->lay.csum);
            cp.sum_gg = cp.sum + (size_t)p.corr_groups * p.corr_levels * p.corr_bins;
            cp.M = p.n_chains; cp.chain_offset = p.chain_offset;
            cp.n_samples = (int)nsmp; cp.L = p.corr_levels; cp.Pb = p.corr_bins; cp.groups = p.corr_groups;
            cp.Mv = (long long)p.n_chains * sp.n_comp;
            std::memcpy(cp.pos, c->cpos, sizeof cp.pos); std::memcpy(cp.filled, c->cfil, sizeof cp.filled);
            std::memcpy(cp.parity, c->cpar, sizeof cp.parity);
            CK(c, launch_corr(cp, c->st));
            c->launches += 1;
            for (long long s = 0; s < nsmp; ++s) corr_schedule_sample(c);
        }
        c->n_records += nrec;
        c->step += T;
        left -= T;
    }
    return SSM_OK;
}

extern "C" int ssm_step(ssm_ctx *c, int64_t n_steps, double shear_rate)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (n_steps < 0) return fail(c, SSM_EINVAL, "n_steps < 0");
    if (!std::isfinite(shear_rate)) return fail(c, SSM_EINVAL, "shear_rate is not finite");
    return step_impl(c, n_steps, shear_rate, nullptr, 1);
}

// number of groups and tiles per group for blocks of chains_per_group local chains; false if a warp tile
// would hold chains of two groups
static bool group_geometry(const ssm_ctx *c, int64_t cpg, long long *n_groups, long long *tiles_per_group)
{
    const long long M = c->p.n_chains, cpw = chains_per_warp(padded_beads(c->p.n_beads));
    if (cpg < 1) return false;
    if (cpg >= M) { *n_groups = 1; *tiles_per_group = c->lay.n_tiles; return true; }
    if (cpg % cpw != 0) return false;
    *n_groups = (M + cpg - 1) / cpg; *tiles_per_group = cpg / cpw;
    return true;
}

extern "C" int ssm_step_kappa(ssm_ctx *c, int64_t n_steps, int64_t chains_per_group, const double *h_kappa)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (n_steps < 0) return fail(c, SSM_EINVAL, "n_steps < 0");
    if (!h_kappa) return fail(c, SSM_EINVAL, "h_kappa is NULL");
    long long ng = 0, tpg = 0;
    if (!group_geometry(c, chains_per_group, &ng, &tpg))
        return fail(c, SSM_EINVAL, "chains_per_group must be >= n_chains (one group) or a multiple of the chains per warp, 256 / (n_beads rounded up to 8, 16, 32, 64 or 128)");
    c->kappa_host.resize((size_t)ng * 9);
    for (size_t i = 0; i < (size_t)ng * 9; ++i) {
        if (!std::isfinite(h_kappa[i])) return fail(c, SSM_EINVAL, "kappa is not finite");
        c->kappa_host[i] = (float)(h_kappa[i] * c->p.dt);
    }
    float *d_kappa = reinterpret_cast<float *>(c->ws + c->lay.kappa);
    CK(c, cudaMemcpyAsync(d_kappa, c->kappa_host.data(), (size_t)ng * 9 * 4, cudaMemcpyHostToDevice, c->st));
    return step_impl(c, n_steps, 0.0, d_kappa, tpg);
}

extern "C" int ssm_step_kappa_device(ssm_ctx *c, int64_t n_steps, int64_t chains_per_group, const double *d_kappa)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (n_steps < 0) return fail(c, SSM_EINVAL, "n_steps < 0");
    if (!d_kappa) return fail(c, SSM_EINVAL, "d_kappa is NULL");
    long long ng = 0, tpg = 0;
    if (!group_geometry(c, chains_per_group, &ng, &tpg))
        return fail(c, SSM_EINVAL, "chains_per_group must be >= n_chains (one group) or a multiple of the chains per warp, 256 / (n_beads rounded up to 8, 16, 32, 64 or 128)");
    float *d_table = reinterpret_cast<float *>(c->ws + c->lay.kappa);
    CK(c, launch_kappa(d_kappa, d_table, ng * 9, c->p.dt, c->st));
    c->launches += 1;
    return step_impl(c, n_steps, 0.0, d_table, tpg);
}

extern "C" int ssm_recenter(ssm_ctx *c)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    CK(c, launch_recenter(c->ws + c->lay.state, c->p.n_beads, c->p.n_chains, c->st));
    c->launches += 1;
    c->low_mode = 0;                       // every low word is zero again
    return SSM_OK;
}

extern "C" int ssm_group_stress_device(ssm_ctx *c, int64_t chains_per_group, double *d_out)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!d_out) return fail(c, SSM_EINVAL, "d_out is NULL");
    if (chains_per_group < 1) return fail(c, SSM_EINVAL, "chains_per_group must be >= 1");
    const long long M = c->p.n_chains, cpg = chains_per_group < M ? chains_per_group : M, ng = (M + cpg - 1) / cpg;
    if ((size_t)ng * 13 * 8 > c->lay.total - c->lay.stage) return fail(c, SSM_ENOMEM, "staging area too small for this many groups");
    long long *d = reinterpret_cast<long long *>(c->ws + c->lay.stage);
    CK(c, cudaMemsetAsync(d, 0, (size_t)ng * 13 * 8, c->st));
    CK(c, launch_group_stress(c->ws + c->lay.state, d, c->p.n_beads, M, cpg, c->sp.cs, c->st));
    CK(c, launch_group_mean(d, d_out, ng, M, cpg, c->st));
    c->launches += 2;
    return SSM_OK;
}

extern "C" int ssm_group_stress(ssm_ctx *c, int64_t chains_per_group, double *h_out)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!h_out) return fail(c, SSM_EINVAL, "h_out is NULL");
    if (chains_per_group < 1) return fail(c, SSM_EINVAL, "chains_per_group must be >= 1");
    const long long M = c->p.n_chains, cpg = chains_per_group < M ? chains_per_group : M, ng = (M + cpg - 1) / cpg;
    if ((size_t)ng * 13 * 8 > c->lay.total - c->lay.stage) return fail(c, SSM_ENOMEM, "staging area too small for this many groups");
    long long *d = reinterpret_cast<long long *>(c->ws + c->lay.stage);
    CK(c, cudaMemsetAsync(d, 0, (size_t)ng * 13 * 8, c->st));
    CK(c, launch_group_stress(c->ws + c->lay.state, d, c->p.n_beads, M, cpg, c->sp.cs, c->st));
    c->launches += 1;
    std::vector<long long> raw((size_t)ng * 13);
    CK(c, cudaMemcpyAsync(raw.data(), d, (size_t)ng * 13 * 8, cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaStreamSynchronize(c->st));
    for (long long g = 0; g < ng; ++g) {
        const long long n = (g + 1) * cpg <= M ? cpg : M - g * cpg;
        for (int t = 0; t < 13; ++t)
            h_out[g * 13 + t] = (double)raw[(size_t)g * 13 + t] / ((double)(1 << kStressShift) * (double)n);
    }
    return SSM_OK;
}

extern "C" int ssm_noise_calibration(const ssm_ctx *c, double *h_out)
{
    if (!c || !h_out) return SSM_EINVAL;
    std::memcpy(h_out, c->calib, sizeof c->calib);
    return SSM_OK;
}

extern "C" int64_t ssm_stress_count(const ssm_ctx *c) { return c ? c->n_records : 0; }
extern "C" int64_t ssm_launch_count(const ssm_ctx *c) { return c ? c->launches : 0; }

extern "C" int ssm_stress_sums(ssm_ctx *c, int64_t first, int64_t n, int64_t *h_out)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (first < 0 || n < 0 || first + n > c->n_records) return fail(c, SSM_ERANGE, "stress samples not recorded");
    if (n == 0) return SSM_OK;
    if (!h_out) return fail(c, SSM_EINVAL, "h_out is NULL");
    CK(c, cudaMemcpyAsync(h_out, c->ws + c->lay.stress + (size_t)first * 96, (size_t)n * 96, cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaStreamSynchronize(c->st));
    return SSM_OK;
}

extern "C" int ssm_stress_sums_device(ssm_ctx *c, int64_t first, int64_t n, int64_t **d_ptr)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!d_ptr) return fail(c, SSM_EINVAL, "d_ptr is NULL");
    if (first < 0 || n < 0 || first + n > c->n_records) return fail(c, SSM_ERANGE, "stress samples not recorded");
    *d_ptr = reinterpret_cast<int64_t *>(c->ws + c->lay.stress) + first * 12;
    return SSM_OK;
}

static int order_streams(ssm_ctx *c, cudaStream_t first, cudaStream_t then)
{
    if (first == then) return SSM_OK;
    cudaEvent_t ev;
    CK(c, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    cudaError_t e = cudaEventRecord(ev, first);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(then, ev, 0);
    cudaEventDestroy(ev);                       // released once the wait has been satisfied
    if (e != cudaSuccess) return cuda_fail(c, e, "stream ordering");
    return SSM_OK;
}

extern "C" int ssm_stream_wait_ctx(ssm_ctx *c, void *cuda_stream)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    return order_streams(c, c->st, (cudaStream_t)cuda_stream);
}

extern "C" int ssm_ctx_wait_stream(ssm_ctx *c, void *cuda_stream)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    return order_streams(c, (cudaStream_t)cuda_stream, c->st);
}

extern "C" int ssm_stress(ssm_ctx *c, int64_t first, int64_t n, double *h_out)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (n > 0 && !h_out) return fail(c, SSM_EINVAL, "h_out is NULL");
    std::vector<int64_t> raw((size_t)(n > 0 ? n : 0) * 12);
    int rc = ssm_stress_sums(c, first, n, raw.data());
    if (rc != SSM_OK) return rc;
    // sums hold sum_bonds (3 b_a b_b - delta_ab) and sum_j ((3/N_s) d_a d_b - delta_ab):
    // sigma_aa = 3 sum b_a^2 - N needs one more -1 per chain (eq 16); sigma^(v) needs none (eq 76)
    static_assert(kStressShift == 18, "ssm_stress_from_sums (ssm_rheo.cu) divides by 2^18");
    if (ssm_stress_from_sums(raw.data(), n, c->p.n_chains, h_out) != SSM_OK) return fail(c, SSM_EINVAL, "bad sample range");
    return SSM_OK;
}

extern "C" int ssm_chain_stress(ssm_ctx *c, float *out, int dev)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!out) return fail(c, SSM_EINVAL, "out is NULL");
    const long long M = c->p.n_chains;
    if (dev) {
        CK(c, launch_chain_stress(c->ws + c->lay.state, out, c->p.n_beads, M, c->sp.cs, c->st));
        c->launches += 1;
        return SSM_OK;
    }
    // host pointer: stage the whole [12][M] array if it fits the staging area, else fail
    if ((size_t)M * 48 > c->lay.total - c->lay.stage) return fail(c, SSM_ENOMEM, "staging area too small for host chain stress");
    float *d = reinterpret_cast<float *>(c->ws + c->lay.stage);
    CK(c, launch_chain_stress(c->ws + c->lay.state, d, c->p.n_beads, M, c->sp.cs, c->st));
    c->launches += 1;
    CK(c, cudaMemcpyAsync(out, d, (size_t)M * 48, cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaStreamSynchronize(c->st));
    return SSM_OK;
}

static int xfer_state_impl(ssm_ctx *c, bool do_export, float *R, float *A, uint8_t *S, int dev)
{
    const int N = c->p.n_beads; const long long M = c->p.n_chains;
    unsigned char *state = c->ws + c->lay.state;
    const int hide = c->low_mode == 2 ? 1 : 0;       // packed low parts are not a float: exported as 0
    int *bad = reinterpret_cast<int *>(c->ws + c->lay.counter) + 2;
    if (dev) {
        CK(c, launch_xfer(do_export, state, R, A, S, N, 0, M, M, hide, bad, c->st));
        c->launches += 1;
        return SSM_OK;
    }
    const long long chunk = c->lay.stage_chains;
    float *dR = reinterpret_cast<float *>(c->ws + c->lay.stage);
    float *dA = dR + (size_t)3 * N * chunk;
    unsigned char *dS = reinterpret_cast<unsigned char *>(dA + (size_t)4 * N * chunk);
    for (long long k0 = 0; k0 < M; k0 += chunk) {
        const long long nk = M - k0 < chunk ? M - k0 : chunk;
        if (do_export) {
            CK(c, launch_xfer(true, state, dR, dA, dS, N, k0, nk, chunk, hide, bad, c->st));
            CK(c, cudaMemcpy2DAsync(R + k0, (size_t)M * 4, dR, (size_t)chunk * 4, (size_t)nk * 4, (size_t)3 * N, cudaMemcpyDeviceToHost, c->st));
            CK(c, cudaMemcpy2DAsync(A + k0, (size_t)M * 4, dA, (size_t)chunk * 4, (size_t)nk * 4, (size_t)4 * N, cudaMemcpyDeviceToHost, c->st));
            CK(c, cudaMemcpy2DAsync(S + k0, (size_t)M, dS, (size_t)chunk, (size_t)nk, (size_t)N, cudaMemcpyDeviceToHost, c->st));
            c->launches += 1;
        } else {
            if (chunk == M) {      // the staging rows are the caller's rows: three plain copies
                CK(c, cudaMemcpyAsync(dR, R, (size_t)M * 4 * 3 * N, cudaMemcpyHostToDevice, c->st));
                CK(c, cudaMemcpyAsync(dA, A, (size_t)M * 4 * 4 * N, cudaMemcpyHostToDevice, c->st));
                CK(c, cudaMemcpyAsync(dS, S, (size_t)M * N, cudaMemcpyHostToDevice, c->st));
            } else {
                CK(c, cudaMemcpy2DAsync(dR, (size_t)chunk * 4, R + k0, (size_t)M * 4, (size_t)nk * 4, (size_t)3 * N, cudaMemcpyHostToDevice, c->st));
                CK(c, cudaMemcpy2DAsync(dA, (size_t)chunk * 4, A + k0, (size_t)M * 4, (size_t)nk * 4, (size_t)4 * N, cudaMemcpyHostToDevice, c->st));
                CK(c, cudaMemcpy2DAsync(dS, (size_t)chunk, S + k0, (size_t)M, (size_t)nk, (size_t)N, cudaMemcpyHostToDevice, c->st));
            }
            CK(c, launch_xfer(false, state, dR, dA, dS, N, k0, nk, chunk, 0, bad, c->st));
            c->launches += 1;
        }
    }
    CK(c, cudaStreamSynchronize(c->st));
    return SSM_OK;
}

// no return while copies from / to the caller's buffers are still in flight, also on failure
static int xfer_state(ssm_ctx *c, bool do_export, float *R, float *A, uint8_t *S, int dev)
{
    const int rc = xfer_state_impl(c, do_export, R, A, S, dev);
    if (rc != SSM_OK) cudaStreamSynchronize(c->st);
    return rc;
}

extern "C" int ssm_get_state(ssm_ctx *c, float *R, float *A, uint8_t *S, int64_t *global_step, int dev)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!R || !A || !S) return fail(c, SSM_EINVAL, "NULL state pointer");
    if (global_step) *global_step = c->step;
    return xfer_state(c, true, R, A, S, dev);
}

// read the "imported state was malformed" flag of the device and clear it; synchronises the stream
static int check_state_flag(ssm_ctx *c)
{
    int bad = 0;
    int *d_bad = reinterpret_cast<int *>(c->ws + c->lay.counter) + 2;
    CK(c, cudaMemcpyAsync(&bad, d_bad, sizeof bad, cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaStreamSynchronize(c->st));
    if (bad) {
        CK(c, cudaMemsetAsync(d_bad, 0, sizeof bad, c->st));
        return fail(c, SSM_EINVAL, "S is malformed: a chain's occupied slots must be its leading ones and hold bead indices 1..n_beads "
                                   "(the offending slots were cleared)");
    }
    return SSM_OK;
}

extern "C" int ssm_set_state(ssm_ctx *c, const float *R, const float *A, const uint8_t *S, int64_t global_step, int dev)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!R || !A || !S) return fail(c, SSM_EINVAL, "NULL state pointer");
    if (global_step < 0) return fail(c, SSM_EINVAL, "global_step < 0");
    int rc = xfer_state(c, false, const_cast<float *>(R), const_cast<float *>(A), const_cast<uint8_t *>(S), dev);
    if (rc != SSM_OK) { c->state_valid = false; return rc; }            // part of the ensemble may be new, part old
    c->step = global_step; c->low_mode = 1;                            // A[3] of the caller is the fp32 low part of x
    c->state_valid = true;
    // the import kernel flags a chain whose S is not "bead indices 1..N in the leading slots, 0 after them".  With host
    // pointers the call has synchronised anyway and reports it now; with device pointers it stays asynchronous and the
    // flag waits on the device for ssm_state_status
    return dev ? SSM_OK : check_state_flag(c);
}

extern "C" int ssm_state_status(ssm_ctx *c)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!c->state_valid) return fail(c, SSM_ESTATE, "a state import failed half way: import a state again");
    return check_state_flag(c);
}

// ssm_set_state from HOST buffers followed by ssm_step, as one pipelined call: the ensemble is uploaded in chunks on a copy
// stream, and a chunk's warp tiles are stepped (all n_steps, launch by launch) as soon as it has landed, while the next
// chunks are still on their way.  Chains are independent (eq 54), and the exact integer record sums do not depend on the
// order in which tiles add to them, so the results are those of ssm_set_state + ssm_step bit for bit.
extern "C" int ssm_step_from_host(ssm_ctx *c, const float *R, const float *A, const uint8_t *S, int64_t global_step,
                                  int64_t n_steps, double shear_rate)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!R || !A || !S) return fail(c, SSM_EINVAL, "NULL state pointer");
    if (global_step < 0 || n_steps < 0) return fail(c, SSM_EINVAL, "global_step or n_steps < 0");
    if (!std::isfinite(shear_rate)) return fail(c, SSM_EINVAL, "shear_rate is not finite");
    const ssm_params &p = c->p;
    if (p.sample_every > 0) return fail(c, SSM_ESTATE, "ssm_step_from_host needs the correlator off (it is fed ensemble-wide after every launch)");
    if (p.stress_every > 0) {
        const long long need = (global_step + n_steps) / p.stress_every - global_step / p.stress_every;
        if (c->n_records + need > p.stress_capacity) return fail(c, SSM_ERANGE, "stress buffer would overflow (stress_capacity)");
    }
    const int N = p.n_beads, npad = padded_beads(N);
    const long long M = p.n_chains, cpw = chains_per_warp(npad);
    if (!c->copy_st) {
        CK(c, cudaStreamCreateWithFlags(&c->copy_st, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CK(c, cudaEventCreateWithFlags(&c->ev_copied[i], cudaEventDisableTiming));
            CK(c, cudaEventCreateWithFlags(&c->ev_free[i], cudaEventDisableTiming));
        }
    }
    // two staging buffers of `chunk` chains each (multiples of 32 chains = whole CTAs of the import kernel and whole tiles)
    long long chunk = (c->lay.stage_chains / 2) / 32 * 32;
    if (chunk < 32) return fail(c, SSM_ENOMEM, "staging area too small to pipeline (stage_chains must be >= 64)");
    {   // about sixteen chunks: the first upload, which nothing overlaps, is a sixteenth of the whole, and a launch still has
        // a few tiles per resident warp (measured on C4: 8 / 16 / 32 / 64 chunks -> 33.0 / 32.4 / 36.7 / 39.9 ms per batch)
        const long long want = ((M + 15) / 16 + 31) / 32 * 32;
        if (want < chunk) chunk = want;
    }
    unsigned char *stage[2] = {c->ws + c->lay.stage, c->ws + c->lay.stage + (size_t)chunk * 29 * npad};
    unsigned char *state = c->ws + c->lay.state;
    int *bad = reinterpret_cast<int *>(c->ws + c->lay.counter) + 2;
    const float gdt = (float)(shear_rate * p.dt);
    // From here on copies from the caller's buffers and kernels are in flight on two streams.  A CUDA error must not
    // return while they still are (the caller would free or reuse R, A, S under the DMA), and it leaves the ensemble
    // part new, part old, some chunks stepped: both streams are drained, the step counter and the records stay as they
    // were, and the ctx refuses to step until a state is imported again (SSM_ESTATE).
#define CKQ(c, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { \
        cudaStreamSynchronize((c)->copy_st); cudaStreamSynchronize((c)->st); (c)->state_valid = false; \
        return cuda_fail((c), e_, #call); } } while (0)
    // everything queued on the ctx's stream so far (it may still read the staging area or the state) comes first
    CKQ(c, cudaEventRecord(c->ev_free[0], c->st));
    CKQ(c, cudaEventRecord(c->ev_free[1], c->st));
    long long j = 0;
    for (long long k0 = 0; k0 < M; k0 += chunk, ++j) {
        const long long nk = M - k0 < chunk ? M - k0 : chunk;
        const int b = (int)(j & 1);
        float *dR = reinterpret_cast<float *>(stage[b]);
        float *dA = dR + (size_t)3 * N * chunk;
        unsigned char *dS = reinterpret_cast<unsigned char *>(dA + (size_t)4 * N * chunk);
        CKQ(c, cudaStreamWaitEvent(c->copy_st, c->ev_free[b], 0));
        CKQ(c, cudaMemcpy2DAsync(dR, (size_t)chunk * 4, R + k0, (size_t)M * 4, (size_t)nk * 4, (size_t)3 * N, cudaMemcpyHostToDevice, c->copy_st));
        CKQ(c, cudaMemcpy2DAsync(dA, (size_t)chunk * 4, A + k0, (size_t)M * 4, (size_t)nk * 4, (size_t)4 * N, cudaMemcpyHostToDevice, c->copy_st));
        CKQ(c, cudaMemcpy2DAsync(dS, (size_t)chunk, S + k0, (size_t)M, (size_t)nk, (size_t)N, cudaMemcpyHostToDevice, c->copy_st));
        CKQ(c, cudaEventRecord(c->ev_copied[b], c->copy_st));
        CKQ(c, cudaStreamWaitEvent(c->st, c->ev_copied[b], 0));
        CKQ(c, launch_xfer(false, state, dR, dA, dS, N, k0, nk, chunk, 0, bad, c->st));
        CKQ(c, cudaEventRecord(c->ev_free[b], c->st));
        c->launches += 1;
        // this chunk's tiles through all n_steps
        const long long t0 = k0 / cpw, t1 = (k0 + nk + cpw - 1) / cpw;
        long long step = global_step, nrec_total = c->n_records, left = n_steps;
        while (left > 0) {
            const int T = next_block(c, step, left);
            long long nrec = 0, nsmp = 0;
            StepParams sp = block_params(c, step, nrec_total, T, &nrec, &nsmp);
            sp.gdt = gdt; sp.kappa = nullptr; sp.tiles_per_group = 1;
            sp.tile_first = (int)t0; sp.n_tiles = (int)(t1 - t0);
            sp.counter_slot = c->sp.counter_slot;
            CKQ(c, launch_step(npad, sp, c->grid, c->st));
            c->sp.counter_slot ^= 1;
            c->launches += 1;
            nrec_total += nrec; step += T; left -= T;
        }
    }
    if (p.stress_every > 0) c->n_records += (global_step + n_steps) / p.stress_every - global_step / p.stress_every;
    c->step = global_step + n_steps;
    c->low_mode = 1;                                                  // A[3] of the caller is the fp32 low part of x
    c->state_valid = true;
    return check_state_flag(c);          // synchronises; SSM_EINVAL if some S was malformed (offending slots cleared, steps run)
#undef CKQ
}

extern "C" int ssm_reset_accumulators(ssm_ctx *c)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    return clear_accumulators(c);
}

extern "C" int ssm_set_fusion(ssm_ctx *c, int32_t t)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (t < 1 || t > kMaxFuse) return fail(c, SSM_EINVAL, "steps_per_launch out of range");
    c->fuse = t;
    return SSM_OK;
}

extern "C" int ssm_issue_rates8(ssm_ctx *c, double *h_cycles)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!h_cycles) return fail(c, SSM_EINVAL, "h_cycles is NULL");
    int dev = 0, sms = 0;
    CK(c, cudaGetDevice(&dev));
    CK(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const size_t need = (size_t)(1 + sms * 512) * sizeof(unsigned);
    if (need > c->lay.total - c->lay.stage) return fail(c, SSM_ENOMEM, "staging area too small for the issue-rate probe");
    CK(c, measure_rates(reinterpret_cast<unsigned *>(c->ws + c->lay.stage), sms, c->st, h_cycles));
    return SSM_OK;
}

extern "C" int ssm_set_grid(ssm_ctx *c, int32_t blocks)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (blocks < 0 || blocks > c->grid_default) return fail(c, SSM_EINVAL, "blocks out of range");
    c->grid = blocks == 0 ? c->grid_default : blocks;
    return SSM_OK;
}

extern "C" int ssm_gt_sums(ssm_ctx *c, double *h_sum, int64_t *h_count)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    const ssm_params &p = c->p;
    if (p.sample_every <= 0) return fail(c, SSM_ESTATE, "correlator is off (sample_every = 0)");
    if (!h_sum || !h_count) return fail(c, SSM_EINVAL, "NULL output");
    const size_t n = (size_t)p.corr_groups * p.corr_levels * p.corr_bins;
    std::vector<long long> raw(n);
    CK(c, cudaMemcpyAsync(raw.data(), c->ws + c->lay.csum, n * 8, cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaStreamSynchronize(c->st));
    // chains per group among the local ones: global index = chain_offset + k, group = (index / 32) % groups
    // (a warp of the correlator kernel, 32 consecutive chains, feeds one group)
    std::vector<long long> per_group((size_t)p.corr_groups, 0);
    {
        const unsigned long long lo = p.chain_offset, hi = p.chain_offset + (unsigned long long)p.n_chains;   // [lo, hi)
        for (unsigned long long b = lo >> 5; (b << 5) < hi; ++b) {
            const unsigned long long b0 = b << 5, b1 = b0 + 32;
            per_group[(size_t)(b % (unsigned)p.corr_groups)] += (long long)((b1 < hi ? b1 : hi) - (b0 > lo ? b0 : lo));
        }
    }
    for (int g = 0; g < p.corr_groups; ++g) {
        const long long ng = per_group[(size_t)g];
        for (int lev = 0; lev < p.corr_levels; ++lev)
            for (int q = 0; q < p.corr_bins; ++q) {
                const size_t i = ((size_t)g * p.corr_levels + lev) * p.corr_bins + q;
                h_sum[i] = (double)raw[i] / 65536.0;
                h_count[i] = c->ccount[(size_t)lev * 32 + q] * ng * (p.corr_components == 3 ? 3 : 1);
            }
    }
    return SSM_OK;
}

extern "C" int ssm_gt_sums_virtual(ssm_ctx *c, double *h_sum_gg)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    const ssm_params &p = c->p;
    if (p.sample_every <= 0) return fail(c, SSM_ESTATE, "correlator is off (sample_every = 0)");
    if (!h_sum_gg) return fail(c, SSM_EINVAL, "NULL output");
    const size_t n = (size_t)p.corr_groups * p.corr_levels * p.corr_bins;
    std::vector<long long> raw(n);
    CK(c, cudaMemcpyAsync(raw.data(), c->ws + c->lay.csum + n * 8, n * 8, cudaMemcpyDeviceToHost, c->st));
    CK(c, cudaStreamSynchronize(c->st));
    for (size_t i = 0; i < n; ++i) h_sum_gg[i] = (double)raw[i] / 65536.0;
    return SSM_OK;
}

// eq (66): dGv(t) = <sv(t) g(0)> / <s(t) g(0)> = (sum_gg - sum_fg) / sum_fg, g = s + sv
extern "C" int ssm_gt_virtual(ssm_ctx *c, int32_t *n_lags, double *h_t, double *h_dgv, double *h_se)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!n_lags || !h_t || !h_dgv) return fail(c, SSM_EINVAL, "NULL output");
    const ssm_params &p = c->p;
    if (p.sample_every <= 0) return fail(c, SSM_ESTATE, "correlator is off (sample_every = 0)");
    const int L = p.corr_levels, Pb = p.corr_bins, Gn = p.corr_groups;
    const size_t n_all = (size_t)Gn * L * Pb;
    std::vector<double> fg(n_all), gg(n_all); std::vector<int64_t> cnt(n_all);
    int rc = ssm_gt_sums(c, fg.data(), cnt.data());
    if (rc == SSM_OK) rc = ssm_gt_sums_virtual(c, gg.data());
    if (rc != SSM_OK) return rc;
    const double base = p.dt * p.sample_every;
    int n = 0;
    for (int lev = 0; lev < L; ++lev)
        for (int q = (lev == 0 ? 0 : Pb / 2); q < Pb; ++q) {
            double sfg = 0.0, sgg = 0.0; int64_t cn = 0;
            for (int g = 0; g < Gn; ++g) {
                const size_t i = ((size_t)g * L + lev) * Pb + q;
                sfg += fg[i]; sgg += gg[i]; cn += cnt[i];
            }
            if (cn == 0) continue;
            if (n >= *n_lags) return fail(c, SSM_ERANGE, "n_lags capacity too small");
            h_t[n] = (double)q * std::ldexp(1.0, lev) * base;
            h_dgv[n] = (sgg - sfg) / sfg;
            if (h_se) {
                double mean = 0.0, var = 0.0; int used = 0;
                for (int g = 0; g < Gn; ++g) {
                    const size_t i = ((size_t)g * L + lev) * Pb + q;
                    if (cnt[i] > 0) { mean += (gg[i] - fg[i]) / fg[i]; ++used; }
                }
                if (used > 1) {
                    mean /= used;
                    for (int g = 0; g < Gn; ++g) {
                        const size_t i = ((size_t)g * L + lev) * Pb + q;
                        if (cnt[i] > 0) { const double v = (gg[i] - fg[i]) / fg[i] - mean; var += v * v; }
                    }
                    h_se[n] = std::sqrt(var / (used - 1) / used);
                } else h_se[n] = NAN;
            }
            ++n;
        }
    *n_lags = n;
    return SSM_OK;
}

extern "C" int ssm_gt(ssm_ctx *c, int32_t *n_lags, double *h_t, double *h_G, double *h_se)
{
    if (!c) return fail(nullptr, SSM_EINVAL, "ctx is NULL");
    if (!n_lags || !h_t || !h_G) return fail(c, SSM_EINVAL, "NULL output");
    const ssm_params &p = c->p;
    if (p.sample_every <= 0) return fail(c, SSM_ESTATE, "correlator is off (sample_every = 0)");
    const int L = p.corr_levels, Pb = p.corr_bins, Gn = p.corr_groups;
    std::vector<double> sum((size_t)Gn * L * Pb); std::vector<int64_t> cnt((size_t)Gn * L * Pb);
    int rc = ssm_gt_sums(c, sum.data(), cnt.data());
    if (rc != SSM_OK) return rc;
    const double base = p.dt * p.sample_every, N = (double)p.n_beads;
    int n = 0;
    for (int lev = 0; lev < L; ++lev)
        for (int q = (lev == 0 ? 0 : Pb / 2); q < Pb; ++q) {
            double s = 0.0; int64_t cn = 0;
            for (int g = 0; g < Gn; ++g) { s += sum[((size_t)g * L + lev) * Pb + q]; cn += cnt[((size_t)g * L + lev) * Pb + q]; }
            if (cn == 0) continue;
            if (n >= *n_lags) return fail(c, SSM_ERANGE, "n_lags capacity too small");
            h_t[n] = (double)q * std::ldexp(1.0, lev) * base;
            h_G[n] = s / ((double)cn * N);            // G/(rho0 kT) = <.>/N  (c0 = rho0/N)
            if (h_se) {
                double mean = 0.0, var = 0.0; int used = 0;
                for (int g = 0; g < Gn; ++g) {
                    const int64_t cg = cnt[((size_t)g * L + lev) * Pb + q];
                    if (cg > 0) { mean += sum[((size_t)g * L + lev) * Pb + q] / ((double)cg * N); ++used; }
                }
                if (used > 1) {
                    mean /= used;
                    for (int g = 0; g < Gn; ++g) {
                        const int64_t cg = cnt[((size_t)g * L + lev) * Pb + q];
                        if (cg > 0) { const double v = sum[((size_t)g * L + lev) * Pb + q] / ((double)cg * N) - mean; var += v * v; }
                    }
                    h_se[n] = std::sqrt(var / (used - 1) / used);
                } else h_se[n] = NAN;
            }
            ++n;
        }
    *n_lags = n;
    return SSM_OK;
}

extern "C" void ssm_destroy(ssm_ctx *c)
{
    if (!c) return;
    if (c->copy_st) {
        cudaStreamSynchronize(c->copy_st);
        for (int i = 0; i < 2; ++i) { cudaEventDestroy(c->ev_copied[i]); cudaEventDestroy(c->ev_free[i]); }
        cudaStreamDestroy(c->copy_st);
    }
    delete c;
}

extern "C" const char *ssm_last_error(const ssm_ctx *c) { return c ? c->err.c_str() : g_err.c_str(); }

// ---------------------------------------------------------------------------------------
// Access for the library's other translation units (ssm_noalloc.cu) to a ctx, whose layout stays private to this file.
// ---------------------------------------------------------------------------------------
namespace ssm {
void ctx_view(const ssm_ctx *c, CtxView *v)
{
    v->state = c->ws + c->lay.state; v->n_beads = c->p.n_beads; v->n_chains = c->p.n_chains; v->cs = c->sp.cs;
    v->stream = c->st;
}
int ctx_fail(ssm_ctx *c, int code, const char *msg) { return fail(c, code, msg); }
void ctx_add_launches(ssm_ctx *c, int n) { c->launches += n; }
}  // namespace ssm
