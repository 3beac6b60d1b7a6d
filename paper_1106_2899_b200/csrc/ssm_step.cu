// ssm_step.cu -- the fused multi-step kernel of the slip-spring ensemble (sm_100a).
//
// One launch advances every chain n_fuse time steps through the three substeps of
// PAPER.md lines 292-347 (section 3.1) with the chain state resident on chip:
//   bead phase  (every lane, 8 beads each): noise w_i (eqs 46, 47), Rouse bond force and
//               slip-spring force (eq 1), explicit Euler (eq 44), bond virial (eq 16);
//   slot phase  (the warp's slip-springs, dealt one per lane over all its chains): anchor
//               advection (eq 45), Glauber hop (eqs 23, 24, 48, 49), destruction (eq 53),
//               virtual stress (eq 76) and the force scatter for the next step;
//               construction attempts (eqs 50-52) are drawn by the chain's bead lanes;
//   reduction   per recorded step, one warp-wide integer add (redux) per stress component
//               into CTA-wide int64 fixed-point accumulators (eq 54), flushed once per CTA.
// Mapping and layouts: ssm_common.h and DESIGN.md section 6.
#include <cuda_runtime.h>

#include <atomic>

#include "ssm_common.h"
#include "ssm_rng.cuh"

namespace ssm {

#define SSM_CAT2(a, b) a##b
#define SSM_CAT(a, b) SSM_CAT2(a, b)

#ifdef SSM_G   // ---- the kernels of one G (this file is compiled once per G, and once without for the dispatcher)

template <int G> struct Log2;
template <> struct Log2<1> { static constexpr int v = 0; };
template <> struct Log2<2> { static constexpr int v = 1; };
template <> struct Log2<4> { static constexpr int v = 2; };
template <> struct Log2<8> { static constexpr int v = 3; };
template <> struct Log2<16> { static constexpr int v = 4; };

__device__ __forceinline__ float mufu_ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

constexpr unsigned kFull = 0xffffffffu;

// Anchor advection under a general velocity gradient (eq 45 with the tensor of eq 21), one coordinate.
// Eq (45) adds nearly the same small increment every step, which a plain fp32 sum rounds the same way
// every step (or drops altogether when it is below half an ulp), so each coordinate is advanced as a
// compensated sum whose low part is kept as a signed 10-bit integer q in units of ulp(hi)/1024 =
// 2^(e - 160), e = biased exponent of hi (three of them share the fourth word of the anchor; layout
// in ssm_common.h).  hi: coordinate, inc: dt (kappa . A) of this coordinate, q: low part in; returns
// the new coordinate and the new low part in q.
__device__ __forceinline__ float advect_packed(float hi, float inc, int &q)
{
    const int e = (__float_as_int(hi) >> 23) & 0xFF;
    const float unit = __int_as_float(max(e - 33, 0) << 23);
    const float t = fmaf((float)q, unit, inc);
    const float sum = hi + t;
    const float bb = sum - hi;
    const float low = (hi - (sum - bb)) + (t - bb);          // hi + t = sum + low exactly (two-sum)
    const int e2 = (__float_as_int(sum) >> 23) & 0xFF;
    const float inv = __int_as_float((287 - max(e2, 34)) << 23);                    // 2^(160 - e2)
    q = e2 >= 34 ? max(-512, min(511, __float2int_rn(low * inv))) : 0;
    return sum;
}

// FLOW: 0 = no flow, 1 = simple shear kappa_xy (eq 60), 2 = one full tensor per group of chains (eqs 18, 21)
// RAGGED: the chain has fewer beads than the 8G places it occupies (ssm_common.h)
template <int G, int FLOW, bool RAGGED>
__global__ void __launch_bounds__(kBlockThreads, 2) ssm_step_kernel(const __grid_constant__ StepParams P)
{
    constexpr bool SHEAR = FLOW == 1;
    constexpr int N = kBPL * G, CPW = 32 / G, LG = Log2<G>::v, LN = LG + 3, WPC = (N + 31) / 32;
    extern __shared__ __align__(16) unsigned char smem[];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int l = lane & (G - 1), cw = lane >> LG;
    // NA = the chain's number of beads; N = 8G places (NA < N: the places NA..N-1 are padding at the origin)
    const int NA = RAGGED ? P.n_act : N;
    constexpr bool ragged = RAGGED;
    const int real_here = min(kBPL, max(0, NA - kBPL * l));          // real beads among this lane's 8 places
    const float bonds_here = (float)min(kBPL, max(0, NA - 1 - kBPL * l));   // bonds i -> i+1 that start in this lane
    unsigned char *wb = smem + warp * kSmWarp;
    // mirror of the bead positions: the lane's 24 register floats as they are (6 x 16 bytes per lane,
    // bead b of the warp at word fx_index(b): the same index as Fx), read by the slot phase as three scalars per bead;
    // lq = the lane's first 16-byte word in it
    const int lq = lane * 6 + (lane >> 2);
    float *Rf = reinterpret_cast<float *>(wb + kSmRm);
    float4 *Rf4 = reinterpret_cast<float4 *>(wb + kSmRm);
    auto bead = [&](int fi) -> float4 { return make_float4(Rf[fi], Rf[fi + 1], Rf[fi + 2], 0.0f); };
    float4 *A4 = reinterpret_cast<float4 *>(wb + kSmA);
    int *Fx = reinterpret_cast<int *>(wb + kSmFx);
    int4 *Fx4 = reinterpret_cast<int4 *>(wb + kSmFx);
    unsigned char *Sb = wb + kSmS;
    int *Zs = reinterpret_cast<int *>(wb + kSmZ);
    int *Xp = reinterpret_cast<int *>(wb + kSmX);
    unsigned *Ev = reinterpret_cast<unsigned *>(wb + kSmEv);
    unsigned *Dm = reinterpret_cast<unsigned *>(wb + kSmDm);
    unsigned char *Map = wb + kSmMap;
    int *Samp = reinterpret_cast<int *>(wb + kSmSamp);
    int *Samp2 = reinterpret_cast<int *>(wb + kSmSamp2);
    float *Kap = reinterpret_cast<float *>(wb + kSmKap);
    int *Stage = reinterpret_cast<int *>(wb + kSmStage);
    int4 *Stage4 = reinterpret_cast<int4 *>(wb + kSmStage);
    unsigned long long *acc = reinterpret_cast<unsigned long long *>(smem + kSmAcc);

#ifdef SSM_CHECK
    // the checked build starts from poisoned shared memory (all bits set: NaN as a float, -1 as an index), so that a
    // read of a word nothing has written shows in the results (tests/test_gpu_sanitize.py compares them with the
    // product build's bit for bit); stands in for compute-sanitizer's initcheck, which this pool does not run
    for (int i = threadIdx.x; i < kSmStep / 4; i += kBlockThreads) reinterpret_cast<unsigned *>(smem)[i] = 0xFFFFFFFFu;
    __syncthreads();
#endif
    const BoxMuller bm_noise(P.bm_noise), bm_anchor(P.bm_anchor);
    // each warp keeps its own copy of the Philox round keys inside its region: their address is then a
    // constant offset from the warp's base register (a CTA-wide copy costs an address computation per call)
    const uint4 *Keys = reinterpret_cast<const uint4 *>(wb + kSmKeys);
    // the launch-constant part of the Philox calls of this tile's chains (ssm_rng.cuh, stream_prefix): [domain][chain]
    constexpr bool PRE = CPW <= 16, PRE_AT = CPW <= 8;      // the table holds 40 entries: three domains of 8 chains, or NOISE and SLOT of 16
    uint4 *Pre = reinterpret_cast<uint4 *>(wb + kSmPre);
    if (lane < 20) reinterpret_cast<unsigned *>(wb + kSmKeys)[lane] = P.rk[lane];
    for (int i = threadIdx.x; i < kMaxFuse * 12; i += kBlockThreads) acc[i] = 0ull;
    Samp[lane] = 0; Samp2[lane] = 0; Samp2[32 + lane] = 0;
    Dm[lane] = 0u;
    Ev[lane] = 0u; Ev[32 + lane] = 0u;      // candidate masks, and the chains' last candidates (taken with atomicMax: must start at 0)
    reinterpret_cast<unsigned *>(Map)[lane] = 0u;
    __syncthreads();

    // dealing: slip-spring f of the warp (0 <= f < Tz) belongs to the chain c with
    // Xp[c] <= f < Xp[c+1] (Xp = exclusive prefix of Z over the warp's chains) and is its slot
    // f - Xp[c]
    auto locate = [&](int f, int &c, int &j) {
        c = 0;
#pragma unroll
        for (int st = CPW / 2; st >= 1; st >>= 1)
            if (f >= Xp[c + st]) c += st;
        j = f - Xp[c];
    };

    // dealing cache: byte it of cj = (c << LN) | j of this lane's slip-spring number lane + 32 it
    // (it = 0..3).  It only changes when some Z of the warp changes.  deal(z) takes the Z of the
    // lane's own chain, forms the prefix over the chains with shuffles (every lane of a chain
    // holds the same z, so a scan over lanes with strides G, 2G, .. is a scan over chains), lets
    // the lanes of a chain write the entries of their chain's slip-springs into Map, and returns
    // the warp's total Tz.  Xp is kept for locate(), which serves slip-springs number >= 128 only.
    unsigned cj = 0u;
    auto deal = [&](int z) -> int {
        int incl = z;
#pragma unroll
        for (int o = G; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(kFull, incl, o);
            if (lane >= o) incl += t;
        }
        const int total = __shfl_sync(kFull, incl, 31);
        const int x0 = incl - z;
        if (l == 0) Xp[cw + 1] = incl;
        if (lane == 0) Xp[0] = 0;
        for (int j = l; j < z; j += G) {
            const int f = x0 + j;
            if (f < 128) Map[((f & 31) << 2) | (f >> 5)] = (unsigned char)((cw << LN) | j);
        }
        __syncwarp();
        cj = reinterpret_cast<const unsigned *>(Map)[lane];
        SSM_ASSERT(z >= 0 && z <= N && total <= 256);
#ifdef SSM_CHECK
        for (int it = 0; it < 4; ++it)
            if (lane + 32 * it < total) {
                const int e = (int)((cj >> (8 * it)) & 0xFFu);
                SSM_ASSERT((e >> LN) < CPW && (e & (N - 1)) < Zs[e >> LN] && Xp[e >> LN] + (e & (N - 1)) == lane + 32 * it);
            }
#endif
        return total;
    };
    // (c << LN) | j of slip-spring number f = lane + 32 it of the warp (f < Tz)
    auto slot_index = [&](int it, int f) -> int {
        if (it < 4) return (int)((cj >> (8 * it)) & 0xFFu);
        int c, j;
        locate(f, c, j);
        return (c << LN) | j;
    };

    // the same for the slip-springs number 128 + lane + 32 q, q = 0..3 (byte q), which only a warp with more than 128
    // slip-springs has: found through the prefix in shared memory
    auto deal_high = [&](int Tz) -> unsigned {
        unsigned hi = 0u;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int f = 128 + lane + 32 * q;
            int c = 0, j = 0;
            if (f < Tz) locate(f, c, j);
            hi |= (unsigned)((c << LN) | j) << (8 * q);
        }
        return hi;
    };

    // add the staged warp sums of records [r0, r1) to the CTA's 64-bit sums
    auto flush_stage = [&](int r0, int r1) {
        __syncwarp();
        for (int i = lane; i < (r1 - r0) * 12; i += 32) {
            const int v = Stage[i];
            if (v != 0) atomicAdd(acc + r0 * 12 + i, (unsigned long long)(long long)v);
        }
        __syncwarp();
    };

    // tiles: every warp starts on its own, the rest are handed out first come, first served (a counter in the
    // workspace), so that a small ensemble, whose tiles per warp are 1 or 2, keeps every SM busy to the end;
    // results do not depend on which warp runs a tile.  This launch's counter was zeroed by the previous one.
    const int nwarps = gridDim.x * kWarpsPerBlock;
    if (blockIdx.x == 0 && threadIdx.x == 0) P.tile_counter[1 - P.counter_slot] = 0;
    int tile = blockIdx.x * kWarpsPerBlock + warp;
    for (; tile < P.n_tiles; tile = nwarps + __shfl_sync(kFull, lane == 0 ? atomicAdd(P.tile_counter + P.counter_slot, 1) : 0, 0)) {
        const long long gtile = (long long)P.tile_first + tile;          // the tile's number in the ensemble
        unsigned char *tp = P.state + gtile * kTileBytes;
        const long long chain_local = gtile * CPW + cw;
        const uint32_t chain0 = (uint32_t)(P.chain_offset + (unsigned long long)gtile * CPW);
        const uint32_t chain = chain0 + (uint32_t)cw;
        const bool valid = chain_local < P.n_chains;

        // ---- load the warp tile: R into registers (+ mirror), A, S, Z into shared memory
        float r[24];
        {
            const float4 *gR = reinterpret_cast<const float4 *>(tp + kTileR);
#pragma unroll
            for (int v = 0; v < 6; ++v) {
                const float4 t = gR[v * 32 + lane];
                r[4 * v] = t.x; r[4 * v + 1] = t.y; r[4 * v + 2] = t.z; r[4 * v + 3] = t.w;
            }
#pragma unroll
            for (int v = 0; v < 7; ++v) Fx4[v * 32 + lane] = make_int4(0, 0, 0, 0);
            const float4 *gA = reinterpret_cast<const float4 *>(tp + kTileA);
#pragma unroll
            for (int v = 0; v < 8; ++v) A4[v * 32 + lane] = gA[v * 32 + lane];
            reinterpret_cast<uint2 *>(Sb)[lane] = reinterpret_cast<const uint2 *>(tp + kTileS)[lane];
            Zs[lane] = reinterpret_cast<const int *>(tp + kTileZ)[lane];
            if (PRE && lane < (PRE_AT ? 3 : 2) * CPW) {
                const StreamKey sk0 = make_stream(P.step0, P.rk);
                const int dom = lane / CPW, c = lane - dom * CPW;
                Pre[lane] = stream_prefix(sk0, P.rk, dom == 0 ? DOM_NOISE : (dom == 1 ? DOM_SLOT : DOM_ATTEMPT), chain0 + (uint32_t)c);
            }
            // dt kappa of the group this warp's chains belong to (a tile never straddles two groups)
            if (FLOW == 2 && lane < 9) Kap[lane] = P.kappa[(gtile / P.tiles_per_group) * 9 + lane];
#pragma unroll
            for (int v = 0; v < 6; ++v) Rf4[lq + v] = make_float4(r[4 * v], r[4 * v + 1], r[4 * v + 2], r[4 * v + 3]);
        }
        __syncwarp();
        int Tz = deal(Zs[cw]);

        // forces of the loaded state: scatter -dt (3/N_s) (R_S - A) of every slip-spring into
        // the fixed-point accumulators of bead S (eq 1; used by the first bead phase)
        if (P.springs_on) {
            for (int it = 0, f = lane; f < Tz; f += 32, ++it) {
                const int sidx = slot_index(it, f), base = sidx & ~(N - 1);
                const int s = Sb[sidx];
                const float4 a = A4[sidx], rb = bead(fx_index(base + s - 1));
                int *fp = Fx + fx_index(base + s - 1);
                atomicAdd(fp, __float2int_rn(-P.fx_scale * (rb.x - a.x)));
                atomicAdd(fp + 1, __float2int_rn(-P.fx_scale * (rb.y - a.y)));
                atomicAdd(fp + 2, __float2int_rn(-P.fx_scale * (rb.z - a.z)));
            }
        }
        __syncwarp();

        int rec = 0, smp = 0;           // records / correlator samples taken so far in this launch
        int stage_base = 0;             // first record whose warp sums are still in the staging rows
        bool rec_prev = false, smp_prev = false;
        float sv[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, cnt = 0.f;   // sum d_a d_b and number of this lane's slip-springs
        for (int n = 0;; ++n) {
            // neighbours across the lane boundary: bead 8l-1 and bead 8l+8 (own end bead at the
            // chain ends, so that the missing bond is zero: free ends, eq 1)
            float bl[3], b[24];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                float lf = r[c], rt = r[21 + c];
                if (G > 1) {
                    const float up = __shfl_up_sync(kFull, r[21 + c], 1, G);
                    const float dn = __shfl_down_sync(kFull, r[c], 1, G);
                    if (l != 0) lf = up;
                    if (l != G - 1) rt = dn;
                }
                bl[c] = r[c] - lf;
#pragma unroll
                for (int k = 0; k < 8; ++k) b[3 * k + c] = (k == 7 ? rt : r[3 * (k + 1) + c]) - r[3 * k + c];
            }
            if (ragged) {
                // free end at bead NA (eq 1): no bond leaves the last real bead, none touches a padding place
#pragma unroll
                for (int k = 0; k < 8; ++k)
                    if (k >= NA - 1 - kBPL * l) { b[3 * k] = 0.f; b[3 * k + 1] = 0.f; b[3 * k + 2] = 0.f; }
                if (real_here == 0) { bl[0] = 0.f; bl[1] = 0.f; bl[2] = 0.f; }
            }

            // ---- observables of the state after step n-1 (eqs 16, 76) and ensemble sums (eq 54)
            if (rec_prev || smp_prev) {
                float v[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    v[0] = fmaf(b[3 * k], b[3 * k], v[0]);
                    v[1] = fmaf(b[3 * k + 1], b[3 * k + 1], v[1]);
                    v[2] = fmaf(b[3 * k + 2], b[3 * k + 2], v[2]);
                    v[3] = fmaf(b[3 * k], b[3 * k + 1], v[3]);
                    v[4] = fmaf(b[3 * k + 1], b[3 * k + 2], v[4]);
                    v[5] = fmaf(b[3 * k + 2], b[3 * k], v[5]);
                }
                if (smp_prev) {
                    // per-chain f = sigma_ab, g = sigma_ab + sigma^(v)_ab for the correlator (eq 43): ab = xy, and
                    // yz, zx as well when the isotropic average is on (history q of the chain at [smp][q][chain])
                    for (int q = 0; q < P.n_comp; ++q) {
                        float f = 3.0f * (q == 0 ? v[3] : (q == 1 ? v[4] : v[5]));
#pragma unroll
                        for (int o = G / 2; o >= 1; o >>= 1) f += __shfl_xor_sync(kFull, f, o);
                        if (l == 0) {
                            int *sp = q == 0 ? Samp + cw : Samp2 + (q - 1) * 32 + cw;
                            const int sx = *sp;
                            *sp = 0;
                            const float g = fmaf(P.cs * (1.0f / (float)(1 << kSampleShift)), (float)sx, f);
                            SSM_ASSERT(smp < kMaxFuse);
                            if (valid && P.samples)
                                P.samples[((long long)smp * P.n_comp + q) * P.n_chains + chain_local] = make_float2(f, g);
                        }
                    }
                    ++smp;
                }
                if (rec_prev) {
                    // this lane's share: sum over its bonds of (3 b_a b_b - delta_ab) and over the
                    // slip-springs it handled of ((3/N_s) d_a d_b - delta_ab)
                    // (scaled by 2^kStressShift here, a power of two: the products are the same numbers)
                    constexpr float scale = (float)(1 << kStressShift);
                    const float s3 = valid ? 3.0f * scale : 0.0f, css = P.cs * scale;
                    const float nb = valid ? bonds_here * scale : 0.0f;
                    const float cnts = cnt * scale;
                    float t[12];
                    t[0] = fmaf(s3, v[0], -nb); t[1] = fmaf(s3, v[1], -nb); t[2] = fmaf(s3, v[2], -nb);
                    t[3] = s3 * v[3]; t[4] = s3 * v[4]; t[5] = s3 * v[5];
                    t[6] = fmaf(css, sv[0], -cnts); t[7] = fmaf(css, sv[1], -cnts); t[8] = fmaf(css, sv[2], -cnts);
                    t[9] = css * sv[3]; t[10] = css * sv[4]; t[11] = css * sv[5];
                    // |off-diagonal| <= half the sum of two diagonals, so the two traces bound all
                    // 12 shares by 256, and a 32-lane sum of shares * 2^18 fits 32 bits
                    const bool big = !(3.0f * (v[0] + v[1] + v[2]) < 240.0f && P.cs * (sv[0] + sv[1] + sv[2]) < 240.0f);
                    SSM_ASSERT(rec < kMaxFuse && rec - stage_base >= 0 && rec - stage_base < kStageSteps && rec < P.n_rec);
                    int4 *row = Stage4 + (rec - stage_base) * 3;
                    if (__any_sync(kFull, big)) {
                        // rare (strongly stretched chains): sum the shares as two 32-bit halves and add
                        // them to the CTA sums directly; the staged row of this record is zero
                        long long mine = 0;
#pragma unroll
                        for (int i = 0; i < 12; ++i) {
                            const long long q = __float2ll_rn(t[i]);
                            const int hi = __reduce_add_sync(kFull, (int)(q >> 16));
                            const int lo = __reduce_add_sync(kFull, (int)(q & 0xFFFF));
                            if (lane == i) mine = ((long long)hi << 16) + (long long)lo;
                        }
                        if (lane < 12) atomicAdd(acc + rec * 12 + lane, (unsigned long long)mine);
                        if (lane < 3) row[lane] = make_int4(0, 0, 0, 0);
                    } else {
                        // one warp-wide integer add per component; lane 0 parks the 12 sums in the
                        // warp's staging rows, which are added to the CTA sums every kStageSteps records
                        int tot[12];
#pragma unroll
                        for (int i = 0; i < 12; ++i) tot[i] = __reduce_add_sync(kFull, __float2int_rn(t[i]));
                        if (lane == 0) {
                            row[0] = make_int4(tot[0], tot[1], tot[2], tot[3]);
                            row[1] = make_int4(tot[4], tot[5], tot[6], tot[7]);
                            row[2] = make_int4(tot[8], tot[9], tot[10], tot[11]);
                        }
                    }
                    ++rec;
                    if (rec - stage_base == kStageSteps) { flush_stage(stage_base, rec); stage_base = rec; }
                }
            }
            if (n == P.n_fuse) break;

            const unsigned long long step = P.step0 + (unsigned long long)n;
            const StreamKey sk = make_stream(step, P.rk);
            const bool record = (P.rec_mask >> n) & 1u;
            const bool sample = (P.smp_mask >> n) & 1u;
            const int Z0 = Zs[cw];

            // ================= bead phase: substep 1 (eq 44) =================
            float kap[9], ox = 0.f, oy = 0.f, oz = 0.f;       // FLOW 2: dt kappa, and the time-t position of the bead in hand
            if (FLOW == 2) {
#pragma unroll
                for (int i = 0; i < 9; ++i) kap[i] = Kap[i];
            }
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                float z8[8];
                if (PRE) {
                    uint32_t w[4];
                    stream_call_pre(sk, Pre[cw], (uint32_t)(3 * l + q), w, Keys);
#pragma unroll
                    for (int e = 0; e < 4; ++e) bm_noise(w[e], z8[2 * e], z8[2 * e + 1]);
                } else normal_call<true>(sk, P.rk, DOM_NOISE, chain, (uint32_t)(3 * l + q), bm_noise, z8, Keys);
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int4 fx = Fx4[lq + 2 * q + h];
                    Fx4[lq + 2 * q + h] = make_int4(0, 0, 0, 0);
                    const int fxa[4] = {fx.x, fx.y, fx.z, fx.w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int f = 8 * q + 4 * h + e, k = f / 3, c = f % 3;
                        const float lap = b[f] - (k == 0 ? bl[c] : b[f - 3]);
                        float inc = fmaf(P.dt3, lap, z8[4 * h + e]);
                        inc = fmaf((float)fxa[e], 1.0f / (float)(1 << kFxShift), inc);
                        if (SHEAR && c == 0) inc = fmaf(P.gdt, r[f + 1], inc);
                        if (FLOW == 2) {
                            // dt (kappa . R_i)_c from the time-t position (x, y, z of a bead are updated in this order)
                            if (c == 0) { ox = r[f]; oy = r[f + 1]; oz = r[f + 2]; }
                            inc = fmaf(kap[3 * c], ox, fmaf(kap[3 * c + 1], oy, fmaf(kap[3 * c + 2], oz, inc)));
                        }
                        r[f] += inc;
                    }
                }
            }
            if (ragged) {
#pragma unroll
                for (int f = 0; f < 24; ++f)
                    if (f >= 3 * real_here) r[f] = 0.0f;
            }
#pragma unroll
            for (int v = 0; v < 6; ++v) Rf4[lq + v] = make_float4(r[4 * v], r[4 * v + 1], r[4 * v + 2], r[4 * v + 3]);
            __syncwarp();

            // ================= slot phase: substeps 2 and 3 =================
#pragma unroll
            for (int t = 0; t < 6; ++t) sv[t] = 0.0f;
            cnt = 0.0f;
            if (P.springs_on) {
                bool event = false;
                // one slip-spring per lane per pass: number f = lane + 32 it of the warp.  (Two or three
                // per lane in one straight-line pass were measured slower: 8.2 and 9.1 ms against 7.7 ms
                // per launch; the extra predicated-off pass costs more than the overlap of the chains wins.)
                const int nit = (Tz + 31) >> 5;
                unsigned cur = cj;                 // byte 0 = this pass's (chain, slot) of the lane
                for (int it = 0; it < nit; ++it) {
                    const int f = lane + 32 * it;
                    const bool act = f < Tz;
                    if (it == 4) cur = deal_high(Tz);
                    const int sx = (int)(cur & 0xFFu), c = sx >> LN, j = sx & (N - 1), base = sx & ~(N - 1);
                    cur >>= 8;
                    uint32_t w[4];
                    if (PRE) stream_call_pre(sk, Pre[CPW + c], (uint32_t)(j >> 1), w, Keys);
                    else stream_call<true>(sk, P.rk, DOM_SLOT, chain0 + (uint32_t)c, (uint32_t)(j >> 1), w, Keys);
                    const uint32_t w_hop = (j & 1) ? w[2] : w[0], w_end = (j & 1) ? w[3] : w[1];
                    SSM_ASSERT(!act || (c < CPW && j < Zs[c] && Sb[sx] >= 1 && Sb[sx] <= NA));
                    const int s = max((int)Sb[sx], 1);       // 1..N (an idle lane may look at an empty slot: any bead will do)
                    float4 a = A4[sx];
                    if (SHEAR) {
                        // eq 45 with kappa_xy only: A_x += dt gamma_dot A_y, as a compensated
                        // (two-sum) update of (A_x, low part): the increment is the same every
                        // step, so a plain fp32 sum would drift linearly instead of randomly
                        const float t = fmaf(P.gdt, a.y, a.w);
                        const float sum = a.x + t;
                        const float bb = sum - a.x;
                        a.w = (a.x - (sum - bb)) + (t - bb);
                        a.x = sum;
                        if (act) A4[sx] = a;
                    }
                    if (FLOW == 2) {
                        // eq 45 with the full tensor; the fourth word holds the three packed low parts
                        const int pw = __float_as_int(a.w);
                        int q0 = (pw << 22) >> 22, q1 = (pw << 12) >> 22, q2 = (pw << 2) >> 22;
                        const float ix = fmaf(Kap[0], a.x, fmaf(Kap[1], a.y, Kap[2] * a.z));
                        const float iy = fmaf(Kap[3], a.x, fmaf(Kap[4], a.y, Kap[5] * a.z));
                        const float iz = fmaf(Kap[6], a.x, fmaf(Kap[7], a.y, Kap[8] * a.z));
                        a.x = advect_packed(a.x, ix, q0);
                        a.y = advect_packed(a.y, iy, q1);
                        a.z = advect_packed(a.z, iz, q2);
                        a.w = __int_as_float((q0 & 0x3FF) | ((q1 & 0x3FF) << 10) | ((q2 & 0x3FF) << 20));
                        if (act) A4[sx] = a;
                    }
                    // Glauber hop (eqs 23, 24 with the cap of eqs 48, 49):
                    // p+- = min{ h [1 - tanh x+-], 1/2 } = min{ 2h / (1 + e^{2 x+-}), 1/2 },
                    // x+- = (3/4N_s)(|R_{s+-1}-A|^2 - |R_s-A|^2)
                    const int b0 = base + s - 1;
                    // neighbours along the chain are 3 floats away (7 across the padding after every 32 beads,
                    // which only chains of more than 32 beads can straddle)
                    const int fi = fx_index(b0);
                    SSM_ASSERT(b0 >= base && b0 < base + N && fi >= 0 && fi + 2 < 800);
                    const int up3 = (G > 4 && (b0 & 31) == 31) ? 7 : 3, dn3 = (G > 4 && (b0 & 31) == 0) ? 7 : 3;
                    const float4 r0 = bead(fi);
                    const float4 rp = bead(fi + (s < NA ? up3 : 0));
                    const float4 rm = bead(fi - (s > 1 ? dn3 : 0));
                    const float d0x = r0.x - a.x, d0y = r0.y - a.y, d0z = r0.z - a.z;
                    const float dpx = rp.x - a.x, dpy = rp.y - a.y, dpz = rp.z - a.z;
                    const float dmx = rm.x - a.x, dmy = rm.y - a.y, dmz = rm.z - a.z;
                    const float e0 = fmaf(d0z, d0z, fmaf(d0y, d0y, d0x * d0x));
                    const float ep = fmaf(dpz, dpz, fmaf(dpy, dpy, dpx * dpx));
                    const float em = fmaf(dmz, dmz, fmaf(dmy, dmy, dmx * dmx));
                    float pp = fminf(__fdividef(P.h2, 1.0f + mufu_ex2(P.q2l * (ep - e0))), 0.5f);
                    float pm = fminf(__fdividef(P.h2, 1.0f + mufu_ex2(P.q2l * (em - e0))), 0.5f);
                    if (s == NA) pp = 0.0f;
                    if (s == 1) pm = 0.0f;
                    const float uu = u23(w_hop);
                    const bool up = uu < pp, dn = !up && uu < pp + pm;
                    const int sn = s + (up ? 1 : 0) - (dn ? 1 : 0);
                    // destruction at the ends (eq 53), integer-domain comparison
                    const bool destroyed = (sn == 1 || sn == NA) && code23(w_end) < P.t_destroy;
                    const bool live = act && !destroyed;
                    if (act && sn != s) Sb[sx] = (unsigned char)sn;
                    if (act && destroyed) {
                        atomicOr(Dm + c * WPC + (j >> 5), 1u << (j & 31));
                        event = true;
                    }
                    // a destroyed slip-spring exerts no force and has no virial
                    if (live) {
                        const float dx = up ? dpx : (dn ? dmx : d0x), dy = up ? dpy : (dn ? dmy : d0y),
                                    dz = up ? dpz : (dn ? dmz : d0z);
                        int *fp = Fx + fi + (up ? up3 : 0) - (dn ? dn3 : 0);
                        SSM_ASSERT(sn >= 1 && sn <= NA && fp == Fx + fx_index(base + sn - 1));
                        atomicAdd(fp, __float2int_rn(-P.fx_scale * dx));
                        atomicAdd(fp + 1, __float2int_rn(-P.fx_scale * dy));
                        atomicAdd(fp + 2, __float2int_rn(-P.fx_scale * dz));
                        sv[0] = fmaf(dx, dx, sv[0]); sv[1] = fmaf(dy, dy, sv[1]); sv[2] = fmaf(dz, dz, sv[2]);
                        sv[3] = fmaf(dx, dy, sv[3]); sv[4] = fmaf(dy, dz, sv[4]); sv[5] = fmaf(dz, dx, sv[5]);
                        cnt += 1.0f;
                        if (sample) {
                            atomicAdd(Samp + c, __float2int_rn(dx * dy * (float)(1 << kSampleShift)));
                            if (P.n_comp == 3) {
                                atomicAdd(Samp2 + c, __float2int_rn(dy * dz * (float)(1 << kSampleShift)));
                                atomicAdd(Samp2 + 32 + c, __float2int_rn(dz * dx * (float)(1 << kSampleShift)));
                            }
                        }
                    }
                }
                // construction attempts (eqs 50, 51), drawn by the chain's own lanes; K = N - Z
                // or a fixed K.  The 23-bit code of attempt k is (h << 7) | e (DESIGN.md
                // reading R22): h is a 16-bit half of ATTEMPT call k>>3, so ONE call per lane covers the
                // chain's K <= 8G attempts; e comes from the ANCHOR call, which only a candidate
                // (h <= (T(2 p_c) - 1) >> 7, about 2e-3 per attempt) ever evaluates.
                {
                    const int empty = NA - Z0;
                    int K = P.k_attempts > 0 ? (P.k_attempts < empty ? P.k_attempts : empty) : empty;
                    if (!valid) K = 0;
                    SSM_ASSERT(K >= 0 && K <= NA && Z0 >= 0 && Z0 <= NA);
                    if (8 * l < K) {
                        uint32_t w[4];
                        if (PRE_AT) stream_call_pre(sk, Pre[2 * CPW + cw], (uint32_t)l, w, Keys);
                        else stream_call<true>(sk, P.rk, DOM_ATTEMPT, chain, (uint32_t)l, w, Keys);
                        const int hmax = P.h_c2[K];
                        const unsigned m2 = __vminu2(__vminu2(w[0], w[1]), __vminu2(w[2], w[3]));
                        if ((int)min(m2 & 0xFFFFu, m2 >> 16) <= hmax) {
                            // the lane's candidates (bit e: attempt 8l + e) and (attempt << 16) | half of its last one
                            unsigned cnd = 0u, last = 0u;
#pragma unroll
                            for (int e = 0; e < 8; ++e) {
                                const unsigned h = (w[e >> 1] >> (16 * (e & 1))) & 0xFFFFu;
                                if (8 * l + e < K && (int)h <= hmax) { cnd |= 1u << e; last = ((unsigned)(8 * l + e) << 16) | h; }
                            }
                            atomicOr(Ev + cw * WPC + (l >> 2), cnd << (8 * (l & 3)));
                            atomicMax(Ev + 32 + cw, last);      // the chain's last candidate and its half (largest attempt wins)
                            event = true;
                        }
                    }
                }
                if (__any_sync(kFull, event)) {
                    __syncwarp();
                    int Zn = Z0;
                    if (l == 0) {
                        // rare path, one lane per chain: re-index the chain's slip-springs so that
                        // they occupy slots 0..Z-1.  Destroyed ones are visited from the
                        // last to the first and replaced by the last one; new ones are appended in
                        // attempt order (reading R21).
                        const int base = cw << LN;
                        bool changed = false;
#pragma unroll
                        for (int wd = WPC - 1; wd >= 0; --wd) {
                            unsigned m = Dm[cw * WPC + wd];
                            if (m) { Dm[cw * WPC + wd] = 0u; changed = true; }
                            while (m) {
                                const int bit = 31 - __clz(m);            // highest slot first
                                m &= ~(1u << bit);
                                const int j = 32 * wd + bit;
                                --Zn;
                                SSM_ASSERT(Zn >= 0 && j <= Zn && j < N);
                                if (j != Zn) { Sb[base + j] = Sb[base + Zn]; A4[base + j] = A4[base + Zn]; }
                                Sb[base + Zn] = 0;
                                A4[base + Zn] = make_float4(0.f, 0.f, 0.f, 0.f);
                            }
                        }
                        const int K0 = P.k_attempts > 0 ? min(P.k_attempts, NA - Z0) : NA - Z0;
#pragma unroll
                        for (int wd = 0; wd < WPC; ++wd) {
                            unsigned m = Ev[cw * WPC + wd];
                            if (m) Ev[cw * WPC + wd] = 0u;
                            while (m) {
                                const int bit = __ffs(m) - 1;
                                m &= m - 1u;
                                const int k = 32 * wd + bit;
                                // the candidate's full code: 16 bits of its ATTEMPT half, 7 bits of ANCHOR word 2
                                uint32_t wa[4];
                                stream_call(sk, P.rk, DOM_ANCHOR, chain, (uint32_t)k, wa);
                                const unsigned cd = Ev[32 + cw];
                                unsigned h = cd & 0xFFFFu;
                                if ((cd >> 16) != (unsigned)k) {       // several candidates in one chain: draw the half again
                                    uint32_t w[4];
                                    stream_call(sk, P.rk, DOM_ATTEMPT, chain, (uint32_t)(k >> 3), w);
                                    h = (w[(k & 7) >> 1] >> (16 * (k & 1))) & 0xFFFFu;
                                }
                                const unsigned code = (h << 7) | (wa[2] >> 25);
                                if (code >= P.t_c2[K0]) continue;
                                const int snew = code < P.t_c1[K0] ? 1 : NA;
                                float z3[3], unused;
                                bm_anchor(wa[0], z3[0], z3[1]);                                       // eq 52
                                bm_anchor(wa[1], z3[2], unused);
                                const float4 rb = bead(fx_index(base + snew - 1));
                                const float4 a = make_float4(rb.x + z3[0], rb.y + z3[1], rb.z + z3[2], 0.0f);
                                SSM_ASSERT(Zn >= 0 && Zn < NA && k < K0);
                                Sb[base + Zn] = (unsigned char)snew;
                                A4[base + Zn] = a;
                                ++Zn;
                                changed = true;
                                const float dx = rb.x - a.x, dy = rb.y - a.y, dz = rb.z - a.z;
                                int *fp = Fx + fx_index(base + snew - 1);
                                atomicAdd(fp, __float2int_rn(-P.fx_scale * dx));
                                atomicAdd(fp + 1, __float2int_rn(-P.fx_scale * dy));
                                atomicAdd(fp + 2, __float2int_rn(-P.fx_scale * dz));
                                sv[0] = fmaf(dx, dx, sv[0]); sv[1] = fmaf(dy, dy, sv[1]); sv[2] = fmaf(dz, dz, sv[2]);
                                sv[3] = fmaf(dx, dy, sv[3]); sv[4] = fmaf(dy, dz, sv[4]); sv[5] = fmaf(dz, dx, sv[5]);
                                cnt += 1.0f;
                                if (sample) {
                                    atomicAdd(Samp + cw, __float2int_rn(dx * dy * (float)(1 << kSampleShift)));
                                    if (P.n_comp == 3) {
                                        atomicAdd(Samp2 + cw, __float2int_rn(dy * dz * (float)(1 << kSampleShift)));
                                        atomicAdd(Samp2 + 32 + cw, __float2int_rn(dz * dx * (float)(1 << kSampleShift)));
                                    }
                                }
                            }
                        }
                        Ev[32 + cw] = 0u;
                        if (changed) Zs[cw] = Zn;
                    }
                    __syncwarp();
                    Tz = deal(__shfl_sync(kFull, Zn, cw << LG));
                }
            }
            __syncwarp();
            rec_prev = record; smp_prev = sample;
        }

        if (rec > stage_base) flush_stage(stage_base, rec);

        // ---- store the warp tile
        {
            float4 *gR = reinterpret_cast<float4 *>(tp + kTileR);
#pragma unroll
            for (int v = 0; v < 6; ++v) gR[v * 32 + lane] = make_float4(r[4 * v], r[4 * v + 1], r[4 * v + 2], r[4 * v + 3]);
            float4 *gA = reinterpret_cast<float4 *>(tp + kTileA);
#pragma unroll
            for (int v = 0; v < 8; ++v) gA[v * 32 + lane] = A4[v * 32 + lane];
            reinterpret_cast<uint2 *>(tp + kTileS)[lane] = reinterpret_cast<const uint2 *>(Sb)[lane];
            reinterpret_cast<int *>(tp + kTileZ)[lane] = Zs[lane];
        }
        __syncwarp();
    }

    // ---- flush: one 64-bit reduction per (record, component) per CTA; integer addition is
    // exact, so the result does not depend on the order in which warps and CTAs arrive
    // (deterministic ensemble sums)
    __syncthreads();
    for (int i = threadIdx.x; i < P.n_rec * 12; i += kBlockThreads) {
        const unsigned long long s = acc[i];
        if (s != 0ull) atomicAdd(reinterpret_cast<unsigned long long *>(P.stress) + i, s);
    }
}

// ---------------------------------------------------------------------------------------
// host-side launcher.  This file is compiled once per G with -DSSM_G=<G> (the kernels of that G:
// 3 flows x full / ragged) and once without (the dispatcher), so that the build runs in parallel.
// ---------------------------------------------------------------------------------------
template <int G, int FLOW, bool RAGGED>
static cudaError_t launch_gfr(const StepParams &p, int grid, cudaStream_t st)
{
    // the attribute belongs to the (function, device) pair: remember per device where it has been set
    static std::atomic<unsigned long long> configured{0ull};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev >= 64 || !((configured.load(std::memory_order_relaxed) >> dev) & 1ull)) {
        e = cudaFuncSetAttribute(ssm_step_kernel<G, FLOW, RAGGED>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmStep);
        if (e != cudaSuccess) return e;
        if (dev < 64) configured.fetch_or(1ull << dev, std::memory_order_relaxed);
    }
    ssm_step_kernel<G, FLOW, RAGGED><<<grid, kBlockThreads, kSmStep, st>>>(p);
    return cudaGetLastError();
}

template <int G, int FLOW>
static cudaError_t launch_gf(const StepParams &p, int grid, cudaStream_t st)
{
    return p.n_act != kBPL * G ? launch_gfr<G, FLOW, true>(p, grid, st) : launch_gfr<G, FLOW, false>(p, grid, st);
}

// the affine term of eqs 44, 45 is compiled in only when a velocity gradient is applied: the full tensor
// when a table of tensors is given, else kappa_xy when the shear rate is not zero
cudaError_t SSM_CAT(launch_step_g, SSM_G)(const StepParams &p, int grid, cudaStream_t st)
{
    if (p.kappa) return launch_gf<SSM_G, 2>(p, grid, st);
    return p.gdt != 0.0f ? launch_gf<SSM_G, 1>(p, grid, st) : launch_gf<SSM_G, 0>(p, grid, st);
}

cudaError_t SSM_CAT(step_occupancy_g, SSM_G)(int *blocks_per_sm)
{
    cudaError_t e = cudaFuncSetAttribute(ssm_step_kernel<SSM_G, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmStep);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, ssm_step_kernel<SSM_G, 2, true>, kBlockThreads, kSmStep);
}

#else   // the dispatcher over the bead places per chain, 8G

#define SSM_DECL(g) cudaError_t launch_step_g##g(const StepParams &, int, cudaStream_t); cudaError_t step_occupancy_g##g(int *);
SSM_DECL(1) SSM_DECL(2) SSM_DECL(4) SSM_DECL(8) SSM_DECL(16)

cudaError_t step_occupancy(int n_places, int *blocks_per_sm)
{
    switch (n_places) {
        case 8: return step_occupancy_g1(blocks_per_sm);
        case 16: return step_occupancy_g2(blocks_per_sm);
        case 32: return step_occupancy_g4(blocks_per_sm);
        case 64: return step_occupancy_g8(blocks_per_sm);
        case 128: return step_occupancy_g16(blocks_per_sm);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_step(int n_places, const StepParams &p, int grid, cudaStream_t st)
{
    switch (n_places) {
        case 8: return launch_step_g1(p, grid, st);
        case 16: return launch_step_g2(p, grid, st);
        case 32: return launch_step_g4(p, grid, st);
        case 64: return launch_step_g8(p, grid, st);
        case 128: return launch_step_g16(p, grid, st);
    }
    return cudaErrorInvalidValue;
}
#endif

}  // namespace ssm
