/*
 * ssm.h -- C ABI of libssm.so: ensemble time-stepping of Uneyama's single-chain
 * slip-spring model (arxiv 1106.2899) on one NVIDIA B200 (sm_100a).
 *
 * P:Lnnn = PAPER.md line nnn.  Units b = kT = zeta = 1.
 *
 * The library advances M independent chains of N beads through the three substeps of
 * P:L292-L347 (section 3.1): explicit Euler for beads and anchors (eqs 44, 45), Glauber
 * hop of every slip-spring (eqs 22-24, 48, 49), construction / destruction at the chain
 * ends (eqs 50-53); it records the ensemble means (eq 54) of the stress tensor
 * (eq 16) and of the virtual stress (eq 76) and feeds a per-chain
 * multi-tau correlator for the relaxation modulus G(t) (eq 43).
 *
 * Conventions
 *  - No torch types, no exceptions, no global state.  Every function returns 0 on
 *    success or a negative SSM_E* code; ssm_last_error() gives the text.
 *  - OWNERSHIP: the caller owns every device byte.  It allocates ONE device workspace of
 *    ssm_workspace_bytes() bytes (256-byte aligned) and passes it with a CUDA stream
 *    handle (cudaStream_t cast to void*; NULL = legacy default stream).  The library owns
 *    only the small host-side ssm_ctx.  The workspace must outlive the ctx.
 *  - All work is enqueued on that stream.  Calls that return data to HOST pointers
 *    synchronise the stream before returning; ssm_step() is asynchronous.
 *  - Pointers are marked (host) or (device); "device" means device memory of the GPU the
 *    workspace lives on.
 *  - There is no CPU fallback: without a CUDA device every call fails with SSM_ECUDA.
 *
 * External state layout ("SoA, chain index fastest", used by get/set state):
 *    R[c][i][k]  float32  c = axis 0..2, i = bead 0..N-1, k = chain 0..M-1   -> R[(c*N+i)*M+k]
 *    A[c][j][k]  float32  c = 0..3: x, y, z and the low part of x; j = slip-spring slot 0..zmax-1
 *                                                                            -> A[(c*zmax+j)*M+k]
 *                         The anchor's x is A[0] + A[3]: under shear the library advects it as a
 *                         compensated sum (eq 45 adds the same increment every step, which a plain
 *                         fp32 sum would round the same way every step).  A[3] = 0 is a valid input,
 *                         and what ssm_get_state returns after ssm_step_kappa (whose low parts are
 *                         kept in another encoding, below one ulp of each coordinate).
 *    S[j][k]     uint8    bead index 1..N of slip-spring j, 0 = empty slot   -> S[j*M+k]
 *  The occupied slots of a chain are always the first Z_k ones (the paper's "indices run
 *  from 1 to Z"); zmax = N (the paper's Z <= N).
 */
#ifndef SSM_H
#define SSM_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    SSM_OK      = 0,
    SSM_EINVAL  = -1,   /* bad parameter / unsupported N                         */
    SSM_ENOMEM  = -2,   /* workspace too small or misaligned                     */
    SSM_ECUDA   = -3,   /* CUDA runtime / launch error (text in ssm_last_error)  */
    SSM_ESTATE  = -4,   /* call out of order                                     */
    SSM_ERANGE  = -5    /* sample range not recorded / capacity exceeded         */
};

typedef struct ssm_ctx ssm_ctx;   /* opaque, host side */

/* Parameters of the model as the paper states them plus bookkeeping. */
typedef struct {
    int32_t  n_beads;         /* N, 2..128.  A chain takes 8, 16, 32, 64 or 128 bead places (the   */
                              /* smallest that holds N; 8 places per lane): N = 10, 20, 40, 80 of   */
                              /* the paper run at the speed of 16, 32, 64, 128                      */
    int64_t  n_chains;        /* M >= 1                                                           */
    double   n_s;             /* slip-spring strength N_s (eq 1)                           */
    double   n_0;             /* beads per slip-spring N_0 (eq 10); <= 0 or inf: no slip-  */
                              /* springs (Rouse limit)                                    */
    double   zeta_s;          /* slip-spring friction zeta_s (eqs 23, 24)                         */
    double   dt;              /* time step Delta t                                                */
    uint64_t seed;            /* Philox4x32-10 key                                                */
    uint64_t chain_offset;    /* global index of local chain 0 (Philox is keyed by the global     */
                              /* chain index, so a shard reproduces its part of the full run)     */
    int32_t  stress_every;    /* record the ensemble stress after every k-th step; 0 = never      */
    int64_t  stress_capacity; /* number of stress samples the workspace can hold                  */
    int32_t  sample_every;    /* feed the G(t) correlator after every k-th step; 0 = off          */
    int32_t  corr_levels;     /* multi-tau levels (16); averaging factor m = 2 fixed              */
    int32_t  corr_bins;       /* bins per level (16), even, <= 32                                 */
    int32_t  corr_groups;     /* chain groups for the standard error (32); group = (chain / 32) % groups */
    int32_t  k_attempts;      /* K of eqs (50), (51), "an integer parameter which can depend on Z"    */
                              /* (P:L328): 0 = K = N - Z (the paper's GPU choice);           */
                              /* k > 0 = K = min(k, N - Z) (k = 1 is the paper's CPU choice)         */
    int32_t  corr_components; /* 0 or 1: the correlator follows sigma_xy (eq 43 as printed); 3: xy, yz and  */
                              /* zx each keep their own history and feed the same sums -- the equilibrium   */
                              /* ensemble is isotropic, so this is the same G(t) from three times the data  */
                              /* (meaningful without flow only)                                             */
    int64_t  stage_chains;    /* chains per chunk of the staging area that ssm_get_state / ssm_set_state use for    */
                              /* HOST pointers (29 x bead places bytes each): 0 = 65536.  n_chains makes a state    */
                              /* transfer three copies and one kernel, which is what lets it overlap the stepping   */
                              /* of another ctx on another stream                                                   */
} ssm_params;

/* Bytes of device workspace ssm_init() needs for these parameters (0 on bad parameters). */
size_t ssm_workspace_bytes(const ssm_params *p);

/* Create a context on (device) workspace and sample the equilibrium ensemble on the GPU
 * (eq 13: Gaussian bonds eq 6, Z ~ Poisson(N/N0) eq 12 clamped at zmax,
 * S uniform eq 14, anchors Gaussian eq 15).  Global step counter = 0, accumulators clear. */
int ssm_init(ssm_ctx **out, const ssm_params *p, void *d_workspace, size_t workspace_bytes,
             void *cuda_stream);

/* Advance every chain n_steps time steps with kappa_xy = shear_rate (simple shear, eq 60
 * P:L410; 0 = no flow).  Asynchronous.  The global step counter (Philox's step coordinate)
 * only increases: step(a); step(b) == step(a+b) bit for bit.  Stress samples are appended
 * after every step whose (1-based) global index is a multiple of stress_every; correlator
 * samples likewise with sample_every.  SSM_ERANGE if the stress buffer would overflow. */
int ssm_step(ssm_ctx *ctx, int64_t n_steps, double shear_rate);

/* As ssm_step, under a general velocity gradient tensor (eqs 18, 21; eqs 44, 45 add
 * dt kappa . R_i and dt kappa . A_j), one tensor per GROUP of chains -- the embedding in a flow solver the
 * paper aims at: group g holds the local chains [g chains_per_group, (g+1) chains_per_group),
 * h_kappa (host) [n_groups][9], n_groups = ceil(n_chains / chains_per_group), row-major kappa_ab =
 * d v_a / d r_b in 1/tau0, constant during the call (the host array may be reused after the call returns).
 * chains_per_group >= n_chains means one group; otherwise it must be a multiple of the chains per warp,
 * 256 / (bead places per chain) (the chains of one warp share a tensor), else SSM_EINVAL.  Asynchronous; stress
 * and correlator samples are recorded as by ssm_step (over the whole ensemble; ssm_group_stress reads the
 * groups).  Anchors are advected
 * as compensated sums in all three coordinates (10 extra bits each, kept in the fourth word of the anchor);
 * that word restarts from zero (a change below one ulp of the anchor) when the flow changes between this
 * call and simple shear, and after ssm_set_state. */
int ssm_step_kappa(ssm_ctx *ctx, int64_t n_steps, int64_t chains_per_group, const double *h_kappa);

/* Means over each group of chains_per_group consecutive local chains (any value >= 1; >= n_chains = one
 * group) of the stress of the CURRENT state and of the number of slip-springs: h_out (host)
 * [n_groups][13] = sigma xx,yy,zz,xy,yz,zx (eq 16), sigma_v likewise (eq 76), <Z> (eq 10 at equilibrium;
 * its steady-state value under flow is what P:L428 prints).  Exact integer sums on the device
 * (deterministic).  Synchronises the stream. */
int ssm_group_stress(ssm_ctx *ctx, int64_t chains_per_group, double *h_out);

/* The same two calls for a flow solver that lives on the GPU: d_kappa (device) [n_groups][9] double is read, and
 * d_out (device) [n_groups][13] double is written, by kernels on the ctx's stream; neither call synchronises, so
 * a coupling loop (tensors in, n micro steps, group stresses out) can be queued without the host in it.  Values
 * are those of the host variants bit for bit.  Non-finite tensors are not checked here. */
int ssm_step_kappa_device(ssm_ctx *ctx, int64_t n_steps, int64_t chains_per_group, const double *d_kappa);
int ssm_group_stress_device(ssm_ctx *ctx, int64_t chains_per_group, double *d_out);

/* ssm_group_stress_device for callers that cannot give the library scratch memory.  Which callers: code that runs
 * inside a host application that owns all of the GPU's memory through its own pool and passes a plug-in nothing but the
 * buffers of its inputs and outputs (a raw cudaMalloc there fails, or takes memory the pool counts as its own); a
 * time-critical coupling loop, where cudaMalloc / cudaFree would stall every stream of the device; and a caller whose
 * workspace staging area -- where ssm_group_stress_device keeps its [groups][13] integer sums -- is in use by a state
 * transfer queued on another stream.  Here those sums live in an array built into the library itself: 416 KiB of device
 * memory that every GPU which loads libssm.so holds until the process ends.  Its size is fixed, so at most
 * SSM_NOALLOC_MAX_GROUPS groups: SSM_ERANGE beyond that (take larger groups, or the _device call).
 * Arguments and results are those of ssm_group_stress_device, bit for bit: d_out (device) [n_groups][13] double is
 * written by kernels on the ctx's stream; no host synchronisation; nothing of the workspace but the chain state is read
 * and nothing of it is written.  The call allocates and frees nothing.
 *  - The GPU that holds the ctx's workspace must be the current device (SSM_EINVAL otherwise).
 *  - The first call on each GPU looks up the array's device address (once per device, thread-safe); make that first call
 *    before any stream capture begins.
 *  - All calls on one GPU share the one array, which each call clears before use.  Calls queued on ONE stream are safe.
 *    Calls whose GPU work can overlap (two ctxs on two streams of the same GPU, or two host threads) race on it and
 *    return garbage: order them yourself, or use ssm_group_stress_device for all but one of them. */
#define SSM_NOALLOC_MAX_GROUPS 4096
int ssm_group_stress_noalloc(ssm_ctx *ctx, int64_t chains_per_group, double *d_out);

/* Translate every chain so that its first bead is at the origin, anchors with it.  Nothing observable changes
 * (the model depends on R_i - R_j and R_S - A only: bonds, hop energies, both stresses); under a flow with a
 * stretching direction the chain's centre drifts as exp(kappa t), and a long run (steady elongation) has to call
 * this every few hundred steps to keep the coordinates within fp32's reach.  The anchors' compensation words
 * restart from zero.  Asynchronous.  (The trajectory after the call differs from the uncentred one by fp32
 * rounding only, but is no longer bit-identical to it.) */
int ssm_recenter(ssm_ctx *ctx);

/* Number of stress samples recorded since init / the last reset. */
int64_t ssm_stress_count(const ssm_ctx *ctx);

/* Ensemble means (eq 54) of sigma (eq 16) and sigma^(v) (eq 76) for samples
 * [first_sample, first_sample + n_samples): h_out (host) [n_samples][12] =
 * sigma xx,yy,zz,xy,yz,zx then sigma_v xx,yy,zz,xy,yz,zx.  Means are over the LOCAL
 * chains; ssm_stress_sums gives the exact integer sums a multi-GPU run all-reduces. */
int ssm_stress(ssm_ctx *ctx, int64_t first_sample, int64_t n_samples, double *h_out);

/* Raw fixed-point sums behind ssm_stress: h_out (host) [n_samples][12] int64, value =
 * sum over local chains of (component + delta_ab) * 2^18 rounded per lane. */
int ssm_stress_sums(ssm_ctx *ctx, int64_t first_sample, int64_t n_samples, int64_t *h_out);

/* The means of ssm_stress from raw sums and the TOTAL number of chains behind them (no ctx, no device work): what a
 * sharded run calls on the all-reduced sums of all its ranks.  h_sums (host) [n_samples][12] int64, h_out (host)
 * [n_samples][12]: sum / (2^18 n_chains_total), the diagonal components of sigma minus 1 (eq 16's -N, of which the
 * sums hold N - 1).  For one context ssm_stress_from_sums(ssm_stress_sums(...), n_chains) == ssm_stress(...). */
int ssm_stress_from_sums(const int64_t *h_sums, int64_t n_samples, int64_t n_chains_total, double *h_out);

/* Device address of those sums for samples [first_sample, first_sample + n_samples): *d_ptr
 * (device) int64 [n_samples][12] inside the caller's workspace, so that a multi-GPU run can
 * all-reduce them in place (NCCL) without a copy.  Work queued on the ctx's stream must be
 * ordered before any use on another stream: ssm_stream_wait_ctx / ssm_ctx_wait_stream below do that
 * without blocking the host.  After an in-place all-reduce the sums are those of ALL ranks: ssm_stress
 * (which divides by the local chain count) no longer applies to those samples -- use ssm_stress_from_sums
 * with the global chain count. */
int ssm_stress_sums_device(ssm_ctx *ctx, int64_t first_sample, int64_t n_samples, int64_t **d_ptr);

/* Cross-stream ordering for the exchange above, with CUDA events (no host synchronisation):
 *  ssm_stream_wait_ctx: work queued LATER on cuda_stream (e.g. NCCL's) waits for everything queued so far on the
 *                       ctx's stream (the step kernels that produce the sums);
 *  ssm_ctx_wait_stream: work queued LATER on the ctx's stream (the next steps, ssm_stress_sums) waits for
 *                       everything queued so far on cuda_stream (the all-reduce).
 * cuda_stream = cudaStream_t cast to void* (NULL = the legacy default stream). */
int ssm_stream_wait_ctx(ssm_ctx *ctx, void *cuda_stream);
int ssm_ctx_wait_stream(ssm_ctx *ctx, void *cuda_stream);

/* Per-chain stresses of the CURRENT state: out [12][M] float32 (component-major, chain
 * fastest), host or device. */
int ssm_chain_stress(ssm_ctx *ctx, float *out, int pointers_are_device);

/* Relaxation modulus from the multi-tau correlator (eq 43; per-chain estimator):
 * on entry *n_lags = capacity of the arrays, on exit the number of lags written.
 * h_lag_time[i] in tau0, h_G[i] = G(t_i)/(rho0 kT), h_se[i] (may be NULL) = standard
 * error over chain groups.  All (host). */
int ssm_gt(ssm_ctx *ctx, int32_t *n_lags, double *h_lag_time, double *h_G, double *h_se);

/* Relative contribution of the virtual stress to the relaxation modulus, eq (66):
 *   dGv(t) = [<sv(t) s(0)> + <sv(t) sv(0)>] / [<s(t) s(0)> + <s(t) sv(0)>],  s = sigma_xy, sv = sigma^(v)_xy,
 * from the same multi-tau correlator (it also keeps the sums of g_new g_old, g = s + sv, so that the
 * numerator is <g(t) g(0)> - <s(t) g(0)>).  Arguments as ssm_gt; h_se = standard error of the ratio
 * over chain groups (may be NULL).  ssm_gt_sums_virtual returns the raw g g sums,
 * h_sum_gg (host) [groups][levels][bins], for a multi-GPU reduction beside ssm_gt_sums. */
int ssm_gt_virtual(ssm_ctx *ctx, int32_t *n_lags, double *h_lag_time, double *h_dgv, double *h_se);
int ssm_gt_sums_virtual(ssm_ctx *ctx, double *h_sum_gg);

/* DIAGNOSTIC: the record of the Box-Muller calibration behind this ctx's thermal noise (eqs 44, 46, 47; DESIGN.md section
 * 8.3).  The kernels draw a normal as r cos(theta), r = sqrt(bm log2 u_a), on 2^16 radius and 2^16 angle codes through the
 * GPU's special-function unit; ssm_init sums the variance this really delivers over all codes and picks the fp32 constant
 * bm whose variance is nearest the exact one (once per device and constant in the process; that first ssm_init
 * synchronises the stream).  h_out (host)[8] = [0] the plain constant -2 ln2 2dt rounded to fp32, [1] the constant in use,
 * [2] relative error of the noise variance with [0], [3] with [1], [4] mean cos^2 - 1/2, [5] mean sin^2 - 1/2 over the
 * angle codes, [6] ulps between [0] and [1], [7] 0.  No device work. */
int ssm_noise_calibration(const ssm_ctx *ctx, double *h_out);

/* DIAGNOSTIC, not part of the hot path (bench.py prints it beside the roofline): cycles per
 * group of instructions per scheduler, measured at the step kernel's residency (4 warps per scheduler):
 * h_cycles (host)[8] = [0] FFMA, [1] LOP3 (ALU pipe), [2] IMAD, [3] IMAD.WIDE + the LOP3 folding its halves,
 * [4] the same + 4 FFMA (they do not hide under the multiply: it holds the issue port), [5] MUFU, [6] I2FP + F2I,
 * [7] the instructions of one Philox round (2 multiplies, 2 LOP3).  Runs short kernels on the ctx's stream, uses the workspace's staging
 * area (nothing of the ensemble is touched) and synchronises.  (The 8 in the name is the length of h_cycles: round 1's
 * ssm_issue_rates wrote 4 doubles, and a caller built against it must fail to link rather than be overrun.) */
int ssm_issue_rates8(ssm_ctx *ctx, double *h_cycles);

/* Host post-processing of a tabulated G(t) (section 4.1); no device work, no ctx.
 * h_t[n_lags] strictly increasing lag times >= 0 (as ssm_gt returns them), h_G[n_lags].  All (host).
 *  ssm_moduli : storage and loss moduli, eqs (55), (56), by the trapezoidal rule the paper names
 *               (P:L392), the integral truncated at the last lag: h_storage[q] = G'(h_omega[q]),
 *               h_loss[q] = G''(h_omega[q]).  (On the lags of ssm_gt, whose spacing doubles from level to level, the
 *               rule follows sin(w t), cos(w t) only while w times the spacing is small at the lags where G still
 *               matters: w up to about 0.1 / tau0 for the entangled chains of the paper.)
 *  ssm_eta_star : dynamic viscosity of eq (64) for the Cox-Merz comparison of eq (63):
 *               h_eta_star[q] = sqrt(G'^2 + G''^2) / w at w = h_omega[q] > 0.  (The printed eq (64) lacks the
 *               1/w; eq (63) cannot hold without it -- for w -> 0 only sqrt(..)/w tends to eta_0.)
 *  ssm_eta0   : zero-shear viscosity, eq (59), trapezoidal rule.
 *  ssm_tau_d  : longest relaxation time, eq (58): -1 / slope of the least-squares line through
 *               ln G(t) over t_lo <= t <= t_hi (points with G <= 0 skipped); SSM_ERANGE if the
 *               window holds fewer than two usable points or the slope is not negative.
 * SSM_EINVAL on NULL pointers, n_lags < 2, lag times not increasing, negative frequencies. */
int ssm_moduli(int32_t n_lags, const double *h_t, const double *h_G, int32_t n_omega, const double *h_omega,
               double *h_storage, double *h_loss);
int ssm_eta_star(int32_t n_lags, const double *h_t, const double *h_G, int32_t n_omega, const double *h_omega,
                 double *h_eta_star);
int ssm_eta0(int32_t n_lags, const double *h_t, const double *h_G, double *h_eta0);
int ssm_tau_d(int32_t n_lags, const double *h_t, const double *h_G, double t_lo, double t_hi, double *h_tau_d);

/* Raw correlator sums for multi-GPU reduction: h_sum (host) [groups][levels][bins] double,
 * h_count (host) [groups][levels][bins] int64. */
int ssm_gt_sums(ssm_ctx *ctx, double *h_sum, int64_t *h_count);

/* Checkpoint: copy the state out / in, in the external SoA layout above.  Buffers are
 * caller-owned; pointers_are_device selects device or host pointers for R, A and S.
 * global_step (host) may be NULL on get.  State + global_step = exact resume. */
int ssm_get_state(ssm_ctx *ctx, float *R, float *A, uint8_t *S, int64_t *global_step,
                  int pointers_are_device);
/* ssm_set_state checks S on the device: a chain's occupied slots must be its leading ones and hold bead indices
 * 1..n_beads.  A chain that breaks this keeps its valid leading slots only, so the state stays safe to step.
 *  - HOST pointers: the call synchronises the stream (it has to, for the copies) and returns SSM_EINVAL for a malformed S.
 *  - DEVICE pointers: the call is asynchronous -- one kernel on the ctx's stream, no host synchronisation -- so that a
 *    device-resident loop (ssm_set_state, ssm_step_kappa_device, ssm_group_stress_device, ...) can be queued without the
 *    host in it.  The verdict on S then waits on the device: ssm_state_status returns it.
 * In both cases the ctx holds the imported state afterwards (offending slots cleared) and global_step is set, also when
 * SSM_EINVAL is reported: the error says "this is not the state you meant", not "nothing happened".  Only a CUDA error
 * half way (SSM_ECUDA) leaves the ensemble undefined; stepping is then refused (SSM_ESTATE) until a state is imported. */
int ssm_set_state(ssm_ctx *ctx, const float *R, const float *A, const uint8_t *S,
                  int64_t global_step, int pointers_are_device);

/* Synchronises the stream and returns SSM_EINVAL if a state imported since the last check had a malformed S (see
 * ssm_set_state; the flag is cleared), SSM_ESTATE if an import failed half way, else SSM_OK. */
int ssm_state_status(ssm_ctx *ctx);

/* ssm_set_state from HOST buffers (pinned, or the copies cannot overlap anything) followed by ssm_step(n_steps,
 * shear_rate), as ONE pipelined call: the ensemble is uploaded in about sixteen chunks on a copy stream of the library's
 * own, and a chunk's chains are stepped through all n_steps as soon as it has landed, while the later chunks are still
 * crossing PCIe.  Chains are independent (eq 54) and the integer record sums do not depend on the order in which
 * chains add to them, so state and stress samples are those of ssm_set_state + ssm_step bit for bit.  The correlator must
 * be off (sample_every = 0; SSM_ESTATE otherwise: it is fed ensemble-wide after every launch).  Uses both halves of the
 * staging area as upload buffers (stage_chains >= 64).  Synchronises before returning; S is validated as by
 * ssm_set_state: on SSM_EINVAL the offending slots were cleared, and the n_steps were run and recorded on that cleared
 * state (chunks are stepped as they land, so the verdict on the last chunk comes after the first has been stepped).
 * On a CUDA error both streams are drained before the call returns (no copy from R, A, S is left in flight), the step
 * counter and the records stay as they were, and the ctx refuses to step (SSM_ESTATE) until a state is imported again. */
int ssm_step_from_host(ssm_ctx *ctx, const float *R, const float *A, const uint8_t *S, int64_t global_step,
                       int64_t n_steps, double shear_rate);

/* Clear the stress samples and the correlator; keep the chains and the step counter. */
int ssm_reset_accumulators(ssm_ctx *ctx);

/* Kernel launches issued so far by this ctx (all kernels of this library). */
int64_t ssm_launch_count(const ssm_ctx *ctx);

/* Set the number of time steps fused per kernel launch (1..32; default 32).  Results do
 * not depend on it. */
int ssm_set_fusion(ssm_ctx *ctx, int32_t steps_per_launch);

/* Set the number of CTAs of the step kernel (1..default; 0 restores the default = as many
 * as are resident at once, 2 per SM).  Results do not depend on it. */
int ssm_set_grid(ssm_ctx *ctx, int32_t blocks);

void ssm_destroy(ssm_ctx *ctx);

/* Text of the last error on this ctx (valid until the next call on it); ctx may be NULL
 * for errors of ssm_init / ssm_workspace_bytes. */
const char *ssm_last_error(const ssm_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* SSM_H */
