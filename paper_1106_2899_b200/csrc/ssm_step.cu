// ssm_step.cu -- the fused multi-step kernel of the slip-spring ensemble (sm_100a).
//
// One launch advances every chain n_fuse time steps through the three substeps of
// PAPER.md lines 292-347 (section 3.1) with the chain state resident on chip:
//   bead phase  (all lanes, 4 beads each): noise w_i (eqs 46, 47), Rouse bond force and
//               slip-spring force (eq 1), explicit Euler (eq 44), bond virial (eq 16);
//   slot phase  (lanes own slip-spring pairs): anchor advection (eq 45), Glauber hop
//               (eqs 23, 24, 48, 49), construction / destruction at the ends (eqs 50-53),
//               virtual stress (eq 76) and the force scatter for the next step;
//   reduction   per recorded step, a fixed-tree warp sum of the 12 stress components into
//               warp-private int64 fixed-point accumulators (eq 54), flushed once per CTA.
// Mapping and layouts: ssm_common.h and DESIGN.md section 6.
#include <cuda_runtime.h>

#include "ssm_common.h"
#include "ssm_rng.cuh"

namespace ssm {

template <int G> struct Log2;
template <> struct Log2<2> { static constexpr int v = 1; };
template <> struct Log2<4> { static constexpr int v = 2; };
template <> struct Log2<8> { static constexpr int v = 3; };
template <> struct Log2<16> { static constexpr int v = 4; };
template <> struct Log2<32> { static constexpr int v = 5; };

// Sum 12 per-lane values over the warp with a fixed tree (recursive halving): on return
// lane L holds in v[0] the warp total of component L>>1 (components 12..15 are padding).
__device__ __forceinline__ void warp_reduce_scatter16(float (&v)[16], int lane)
{
#pragma unroll
    for (int h = 8; h >= 1; h >>= 1) {
        const bool up = (lane & (2 * h)) != 0;
#pragma unroll
        for (int i = 0; i < h; ++i) {
            const float send = up ? v[i] : v[i + h];
            const float keep = up ? v[i + h] : v[i];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, 2 * h);
        }
    }
    v[0] += __shfl_xor_sync(0xffffffffu, v[0], 1);
}

template <int G>
__global__ void __launch_bounds__(kBlockThreads, 3) ssm_step_kernel(const __grid_constant__ StepParams P)
{
    constexpr int N = 4 * G, ZMAX = N, CPW = 32 / G;
    constexpr unsigned GMASK = (G == 32) ? 0xffffffffu : ((1u << G) - 1u);
    extern __shared__ __align__(16) unsigned char smem[];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int l = lane & (G - 1), cw = lane >> Log2<G>::v, lane0 = lane - l;
    unsigned char *wb = smem + warp * kSmWarp;
    float *Rl = reinterpret_cast<float *>(wb + kSmRm) + lane * 12;     // this lane's 4 beads
    int *Fl = reinterpret_cast<int *>(wb + kSmFx) + lane * 12;
    float *Rc = reinterpret_cast<float *>(wb + kSmRm) + lane0 * 12;    // this lane's chain
    int *Fc = reinterpret_cast<int *>(wb + kSmFx) + lane0 * 12;
    float *Ac = reinterpret_cast<float *>(wb + kSmA) + cw * ZMAX * 3;
    unsigned char *Sc = wb + kSmS + cw * ZMAX;
    int *Zw = reinterpret_cast<int *>(wb + kSmZ);
    unsigned char *attc = wb + kSmAtt + cw * ZMAX;
    long long *acc = reinterpret_cast<long long *>(smem + kSmAcc) + warp * (kMaxFuse * 12);

    for (int i = lane; i < kMaxFuse * 12; i += 32) acc[i] = 0;
    reinterpret_cast<unsigned *>(wb + kSmAtt)[lane] = 0u;
    __syncwarp();

    const int nwarps = gridDim.x * kWarpsPerBlock;
    for (int tile = blockIdx.x * kWarpsPerBlock + warp; tile < P.n_tiles; tile += nwarps) {
        unsigned char *tp = P.state + (long long)tile * kTileBytes;
        const long long chain_local = (long long)tile * CPW + cw;
        const uint32_t chain = (uint32_t)(P.chain_offset + (unsigned long long)chain_local);
        const float valid = chain_local < P.n_chains ? 1.0f : 0.0f;

        // ---- load the warp tile: R into registers (+ mirror), A, S, Z into shared memory
        float r[12];
        {
            const float4 *gR = reinterpret_cast<const float4 *>(tp + kTileR);
#pragma unroll
            for (int v = 0; v < 3; ++v) {
                const float4 t = gR[v * 32 + lane];
                r[4 * v] = t.x; r[4 * v + 1] = t.y; r[4 * v + 2] = t.z; r[4 * v + 3] = t.w;
                reinterpret_cast<float4 *>(Rl)[v] = t;
                reinterpret_cast<int4 *>(Fl)[v] = make_int4(0, 0, 0, 0);
            }
            const float4 *gA = reinterpret_cast<const float4 *>(tp + kTileA);
            float4 *sA = reinterpret_cast<float4 *>(wb + kSmA);
#pragma unroll
            for (int v = 0; v < 3; ++v) sA[v * 32 + lane] = gA[v * 32 + lane];
            reinterpret_cast<unsigned *>(wb + kSmS)[lane] = reinterpret_cast<const unsigned *>(tp + kTileS)[lane];
            if (lane < 16) Zw[lane] = reinterpret_cast<const int *>(tp + kTileZ)[lane];
        }
        __syncwarp();
        int Zc = Zw[cw];

        // neighbours across the lane boundary: bead 4l-1 and bead 4l+4 (own end bead at the
        // chain ends, so that the missing bond contributes zero: free ends, eq 1)
        float left[3], right[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float up = __shfl_up_sync(0xffffffffu, r[9 + c], 1, G);
            const float dn = __shfl_down_sync(0xffffffffu, r[c], 1, G);
            left[c] = (l == 0) ? r[c] : up;
            right[c] = (l == G - 1) ? r[9 + c] : dn;
        }

        float sv[6];   // virtual-stress partial of this lane's slip-springs (eq 76)

        // slip-spring bookkeeping shared by the prologue and by every step: for the lane's
        // own slots, d = R_S - A; scatter -dt (3/N_s) d into the fixed-point force
        // accumulators of bead S (used by the NEXT bead phase) and sum the virial.
        auto scatter_and_virial = [&]() {
#pragma unroll
            for (int t = 0; t < 6; ++t) sv[t] = 0.0f;
            for (int j0 = 2 * l; j0 < Zc; j0 += 2 * G) {
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int j = j0 + e;
                    if (j < Zc) {
                        const int s = Sc[j] - 1;
                        float d[3];
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            d[c] = Rc[3 * s + c] - Ac[3 * j + c];
                            atomicAdd(&Fc[3 * s + c], __float2int_rn(-P.fx_scale * d[c]));
                        }
                        sv[0] += fmaf(P.cs * d[0], d[0], -1.0f);
                        sv[1] += fmaf(P.cs * d[1], d[1], -1.0f);
                        sv[2] += fmaf(P.cs * d[2], d[2], -1.0f);
                        sv[3] = fmaf(P.cs * d[0], d[1], sv[3]);
                        sv[4] = fmaf(P.cs * d[1], d[2], sv[4]);
                        sv[5] = fmaf(P.cs * d[2], d[0], sv[5]);
                    }
                }
            }
        };
        if (P.springs_on) scatter_and_virial();
        __syncwarp();

        int rec = 0, smp = 0;   // records / correlator samples taken so far in this launch
        for (int n = 0; n < P.n_fuse; ++n) {
            const unsigned long long step = P.step0 + (unsigned long long)n;
            const StreamKey sk = make_stream(P.key0, P.key1, step);

            // ================= bead phase: substep 1 (eq 44) =================
            float z[12];
#pragma unroll
            for (int q = 0; q < 3; ++q) {
                float z4[4];
                normal_call(sk, DOM_NOISE, chain, (uint32_t)(3 * l + q), z4);
                z[4 * q] = z4[0]; z[4 * q + 1] = z4[1]; z[4 * q + 2] = z4[2]; z[4 * q + 3] = z4[3];
            }
            int fx[12];
#pragma unroll
            for (int v = 0; v < 3; ++v) {
                const int4 t = reinterpret_cast<int4 *>(Fl)[v];
                fx[4 * v] = t.x; fx[4 * v + 1] = t.y; fx[4 * v + 2] = t.z; fx[4 * v + 3] = t.w;
                reinterpret_cast<int4 *>(Fl)[v] = make_int4(0, 0, 0, 0);
            }
            float rn[12];
#pragma unroll
            for (int b = 0; b < 4; ++b)
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const float x = r[3 * b + c];
                    const float prev = (b == 0) ? left[c] : r[3 * (b - 1) + c];
                    const float next = (b == 3) ? right[c] : r[3 * (b + 1) + c];
                    float inc = fmaf(P.dt3, (next - x) - (x - prev), P.sq2dt * z[3 * b + c]);
                    inc = fmaf((float)fx[3 * b + c], 1.0f / (float)(1 << kFxShift), inc);
                    if (c == 0) inc = fmaf(P.gdt, r[3 * b + 1], inc);
                    rn[3 * b + c] = x + inc;
                }
#pragma unroll
            for (int i = 0; i < 12; ++i) r[i] = rn[i];
#pragma unroll
            for (int v = 0; v < 3; ++v)
                reinterpret_cast<float4 *>(Rl)[v] = make_float4(r[4 * v], r[4 * v + 1], r[4 * v + 2], r[4 * v + 3]);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float up = __shfl_up_sync(0xffffffffu, r[9 + c], 1, G);
                const float dn = __shfl_down_sync(0xffffffffu, r[c], 1, G);
                left[c] = (l == 0) ? r[c] : up;
                right[c] = (l == G - 1) ? r[9 + c] : dn;
            }
            __syncwarp();

            const unsigned long long done = step + 1ull;
            const bool record = P.stress_every > 0 && done % (unsigned)P.stress_every == 0;
            const bool sample = P.sample_every > 0 && done % (unsigned)P.sample_every == 0;

            // ================= slot phase: substeps 2 and 3 =================
            if (P.springs_on) {
                const int Z0 = Zc;
                bool event = false;
                for (int j0 = 2 * l; j0 < Z0; j0 += 2 * G) {
                    uint32_t w[4];
                    stream_call(sk, DOM_SLOT, chain, (uint32_t)(j0 >> 1), w);
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int j = j0 + e;
                        if (j < Z0) {
                            int s = Sc[j];                                   // 1..N
                            float a[3] = {Ac[3 * j], Ac[3 * j + 1], Ac[3 * j + 2]};
                            if (P.gdt != 0.0f) {                             // eq 45, kappa_xy only
                                a[0] = fmaf(P.gdt, a[1], a[0]);
                                Ac[3 * j] = a[0];
                            }
                            // Glauber hop (eqs 23, 24 with the cap of eqs 48, 49):
                            // p+- = min{ h [1 - tanh x+-], 1/2 } = min{ 2h / (1 + e^{2 x+-}), 1/2 },
                            // x+- = (3/4N_s)(|R_{s+-1}-A|^2 - |R_s-A|^2)
                            //     = (3/4N_s)(R_{s+-1}-R_s).(R_{s+-1}+R_s-2A)   (no cancellation)
                            const int sp = s < N ? s : s - 1, sm = s > 1 ? s - 2 : s - 1;   // 0-based, clamped
                            float dp = 0.0f, dm = 0.0f;
#pragma unroll
                            for (int c = 0; c < 3; ++c) {
                                const float r0 = Rc[3 * (s - 1) + c], rp = Rc[3 * sp + c], rm = Rc[3 * sm + c];
                                const float two_a = 2.0f * a[c];
                                dp = fmaf(rp - r0, (rp + r0) - two_a, dp);
                                dm = fmaf(rm - r0, (rm + r0) - two_a, dm);
                            }
                            float pp = fminf(__fdividef(P.h2, 1.0f + exp2f(P.q2l * dp)), 0.5f);
                            float pm = fminf(__fdividef(P.h2, 1.0f + exp2f(P.q2l * dm)), 0.5f);
                            if (s == N) pp = 0.0f;
                            if (s == 1) pm = 0.0f;
                            const float u = u23(w[2 * e]);
                            if (u < pp) s += 1;
                            else if (u < pp + pm) s -= 1;
                            // destruction at the ends (eq 53), integer-domain comparison
                            const bool destroyed = (s == 1 || s == N) && code23(w[2 * e + 1]) < P.t_destroy;
                            Sc[j] = (unsigned char)(destroyed ? 0xFF : s);     // 0xFF = destroyed marker (N <= 128)
                            event |= destroyed;
                        }
                    }
                }
                // construction attempts (eqs 50, 51): K = number of empty slots, attempt k
                // uses word k&3 of call k>>2
                const int K = ZMAX - Z0;
                if (4 * l < K) {
                    uint32_t w[4];
                    stream_call(sk, DOM_ATTEMPT, chain, (uint32_t)l, w);
                    const unsigned t1 = P.t_c1[K], t2 = P.t_c2[K];
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int k = 4 * l + e;
                        const unsigned code = code23(w[e]);
                        if (k < K && code < t2) {
                            attc[k] = (unsigned char)(code < t1 ? 1 : N);
                            event = true;
                        }
                    }
                }
                const unsigned ev = __ballot_sync(0xffffffffu, event);
                __syncwarp();
                if (((ev >> lane0) & GMASK) != 0u && l == 0) {
                    // rare path: re-index the chain's slip-springs as the paper does:
                    // survivors keep their order, new ones are appended in attempt order
                    int Zs = 0;
                    for (int j = 0; j < Z0; ++j) {
                        const int s = Sc[j];
                        if (s != 0xFF) {
                            if (Zs != j) {
                                Sc[Zs] = (unsigned char)s;
                                Ac[3 * Zs] = Ac[3 * j]; Ac[3 * Zs + 1] = Ac[3 * j + 1]; Ac[3 * Zs + 2] = Ac[3 * j + 2];
                            }
                            ++Zs;
                        }
                    }
                    for (int k = 0; k < K; ++k) {
                        const int snew = attc[k];
                        if (snew) {
                            attc[k] = 0;
                            float z4[4];
                            normal_call(sk, DOM_ANCHOR, chain, (uint32_t)k, z4);   // eq 52
                            Sc[Zs] = (unsigned char)snew;
#pragma unroll
                            for (int c = 0; c < 3; ++c) Ac[3 * Zs + c] = fmaf(P.sq_ns3, z4[c], Rc[3 * (snew - 1) + c]);
                            ++Zs;
                        }
                    }
                    for (int j = Zs; j < Z0; ++j) { Sc[j] = 0; Ac[3 * j] = 0.0f; Ac[3 * j + 1] = 0.0f; Ac[3 * j + 2] = 0.0f; }
                    Zw[cw] = Zs;
                }
                __syncwarp();
                Zc = Zw[cw];
                scatter_and_virial();
                __syncwarp();
            }

            // ================= observables (eqs 16, 76) and ensemble sums (eq 54) =================
            if (record || sample) {
                float v[16];
#pragma unroll
                for (int t = 0; t < 6; ++t) v[t] = 0.0f;
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    float bd[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) bd[c] = ((b == 3) ? right[c] : r[3 * (b + 1) + c]) - r[3 * b + c];
                    v[0] = fmaf(3.0f * bd[0], bd[0], v[0]);
                    v[1] = fmaf(3.0f * bd[1], bd[1], v[1]);
                    v[2] = fmaf(3.0f * bd[2], bd[2], v[2]);
                    v[3] = fmaf(3.0f * bd[0], bd[1], v[3]);
                    v[4] = fmaf(3.0f * bd[1], bd[2], v[4]);
                    v[5] = fmaf(3.0f * bd[2], bd[0], v[5]);
                }
                const float nb = (l == G - 1) ? 3.0f : 4.0f;       // real bonds of this lane: -1 each (eq 16: -N kT 1, +1 on host)
                v[0] -= nb; v[1] -= nb; v[2] -= nb;
#pragma unroll
                for (int t = 0; t < 6; ++t) v[6 + t] = P.springs_on ? sv[t] : 0.0f;
                if (sample) {
                    // per-chain f = sigma_xy, g = sigma_xy + sigma^(v)_xy for the correlator (eq 43)
                    float f = v[3], g = v[3] + v[9];
#pragma unroll
                    for (int o = G / 2; o >= 1; o >>= 1) {
                        f += __shfl_xor_sync(0xffffffffu, f, o);
                        g += __shfl_xor_sync(0xffffffffu, g, o);
                    }
                    if (l == 0 && valid != 0.0f && P.samples)
                        P.samples[(long long)smp * P.n_chains + chain_local] = make_float2(f, g);
                    ++smp;
                }
                if (record) {
#pragma unroll
                    for (int t = 0; t < 12; ++t) v[t] *= valid;
                    v[12] = v[13] = v[14] = v[15] = 0.0f;
                    warp_reduce_scatter16(v, lane);
                    if ((lane & 1) == 0 && lane < 24)
                        acc[rec * 12 + (lane >> 1)] += __float2ll_rn(v[0] * (float)(1 << kStressShift));
                    ++rec;
                }
            }
        }

        // ---- store the warp tile
        {
            float4 *gR = reinterpret_cast<float4 *>(tp + kTileR);
#pragma unroll
            for (int v = 0; v < 3; ++v) gR[v * 32 + lane] = make_float4(r[4 * v], r[4 * v + 1], r[4 * v + 2], r[4 * v + 3]);
            float4 *gA = reinterpret_cast<float4 *>(tp + kTileA);
            const float4 *sA = reinterpret_cast<const float4 *>(wb + kSmA);
#pragma unroll
            for (int v = 0; v < 3; ++v) gA[v * 32 + lane] = sA[v * 32 + lane];
            reinterpret_cast<unsigned *>(tp + kTileS)[lane] = reinterpret_cast<const unsigned *>(wb + kSmS)[lane];
            if (lane < 16) reinterpret_cast<int *>(tp + kTileZ)[lane] = Zw[lane];
        }
        __syncwarp();
    }

    // ---- flush: sum the 8 warps' accumulators in fixed order, one 64-bit reduction per
    // (record, component) per CTA; integer addition is exact, so the result does not depend
    // on the order in which CTAs arrive (deterministic ensemble sums)
    __syncthreads();
    if (P.stress_every > 0) {
        const unsigned long long first = P.step0 / (unsigned)P.stress_every;
        const unsigned long long last = (P.step0 + (unsigned long long)P.n_fuse) / (unsigned)P.stress_every;
        const int nrec = (int)(last - first);
        const long long *a0 = reinterpret_cast<const long long *>(smem + kSmAcc);
        for (int i = threadIdx.x; i < nrec * 12; i += kBlockThreads) {
            long long s = 0;
#pragma unroll
            for (int w = 0; w < kWarpsPerBlock; ++w) s += a0[w * (kMaxFuse * 12) + i];
            if (s != 0) atomicAdd(reinterpret_cast<unsigned long long *>(P.stress) + i, (unsigned long long)s);
        }
    }
}

// ---------------------------------------------------------------------------------------
// host-side launcher
// ---------------------------------------------------------------------------------------
template <int G>
static cudaError_t launch_g(const StepParams &p, int grid, cudaStream_t st)
{
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(ssm_step_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmStep);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    ssm_step_kernel<G><<<grid, kBlockThreads, kSmStep, st>>>(p);
    return cudaGetLastError();
}

template <int G>
static cudaError_t occupancy_g(int *blocks_per_sm)
{
    cudaError_t e = cudaFuncSetAttribute(ssm_step_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmStep);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, ssm_step_kernel<G>, kBlockThreads, kSmStep);
}

cudaError_t step_occupancy(int n_beads, int *blocks_per_sm)
{
    switch (n_beads) {
        case 8: return occupancy_g<2>(blocks_per_sm);
        case 16: return occupancy_g<4>(blocks_per_sm);
        case 32: return occupancy_g<8>(blocks_per_sm);
        case 64: return occupancy_g<16>(blocks_per_sm);
        case 128: return occupancy_g<32>(blocks_per_sm);
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_step(int n_beads, const StepParams &p, int grid, cudaStream_t st)
{
    switch (n_beads) {
        case 8: return launch_g<2>(p, grid, st);
        case 16: return launch_g<4>(p, grid, st);
        case 32: return launch_g<8>(p, grid, st);
        case 64: return launch_g<16>(p, grid, st);
        case 128: return launch_g<32>(p, grid, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace ssm
