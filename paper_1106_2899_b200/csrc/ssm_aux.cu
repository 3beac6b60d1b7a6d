// ssm_aux.cu -- the kernels around the fused step kernel: equilibrium sampler (ssm_init),
// state import / export (ssm_set_state / ssm_get_state), per-chain stress, and the
// per-chain multi-tau correlator that turns (sigma_xy, sigma_xy + sigma^(v)_xy) samples
// into the sums behind G(t) (eq 43).
#include <cuda_runtime.h>

#include <atomic>

#include "ssm_common.h"
#include "ssm_rng.cuh"

namespace ssm {

// ---------------------------------------------------------------------------------------
// Equilibrium sampler, PAPER.md lines 351-355 (eq 13): one thread per chain.
//   1. Gaussian bonds, variance b^2/3 per axis (eq 6); R_1 = 0
//   2. Z ~ Poisson(N/N0) (eq 12) by inversion against integer CDF thresholds, clamped at zmax
//   3. S_j uniform on 1..N (eq 14), A_j Gaussian about R_{S_j}, variance N_s/3 per axis (eq 15)
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) ssm_init_kernel(const __grid_constant__ InitParams P)
{
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= P.n_chains_padded) return;
    const int N = P.n_beads, NP = P.n_pad, zmax = N;
    const uint32_t chain = (uint32_t)(P.chain_offset + (unsigned long long)k);
    const StreamKey sk = make_stream(0ull, P.rk);
    const BoxMuller bm_bond(P.bm_bond), bm_anchor(P.bm_anchor);
    unsigned char *st = P.state;

    float R[128 * 3];
    R[0] = R[1] = R[2] = 0.0f;
    float z8[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    for (int m = 0; m < 3 * (N - 1); ++m) {               // normal m = 3*bond + axis = normal m&7 of call m>>3
        if ((m & 7) == 0) normal_call(sk, P.rk, DOM_INIT_BOND, chain, (uint32_t)(m >> 3), bm_bond, z8);
        R[m + 3] = R[m] + z8[m & 7];
    }
    for (int i = 0; i < N; ++i)
        for (int c = 0; c < 3; ++c) *reinterpret_cast<float *>(st + off_R(k, NP, i, c)) = R[3 * i + c];

    // the chains that pad the last warp tile never carry slip-springs (the step kernel gives them no
    // construction attempts either), so that the warp's slot phase only ever sees real ones
    int Z = 0;
    if (P.springs_on && k < P.n_chains) {
        uint32_t w[4];
        stream_call(sk, P.rk, DOM_INIT_Z, chain, 0u, w);
        const uint32_t code = code23(w[0]);
        while (Z < zmax && code >= P.t_cdf[Z]) ++Z;
    }
    *reinterpret_cast<int *>(st + off_Z(k, NP)) = Z;
    for (int j = 0; j < zmax; ++j) {
        int s = 0; float a[4] = {0.f, 0.f, 0.f, 0.f};
        if (j < Z) {
            uint32_t w[4];
            stream_call(sk, P.rk, DOM_INIT_SLOT, chain, (uint32_t)j, w);
            s = 1 + (int)__umulhi(w[0], (uint32_t)N);
            float z3[3];
            anchor_normals(sk, P.rk, DOM_INIT_ANCHOR, chain, (uint32_t)j, bm_anchor, z3);
            for (int c = 0; c < 3; ++c) a[c] = R[3 * (s - 1) + c] + z3[c];
        }
        st[off_S(k, NP, j)] = (unsigned char)s;
        for (int c = 0; c < 4; ++c) *reinterpret_cast<float *>(st + off_A(k, NP, j, c)) = a[c];
    }
}

cudaError_t launch_init(const InitParams &p, cudaStream_t st)
{
    const int threads = 128;
    const long long blocks = (p.n_chains_padded + threads - 1) / threads;
    ssm_init_kernel<<<(unsigned)blocks, threads, 0, st>>>(p);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// State export / import between the tiled image and the external SoA layout of ssm.h.
// rows 0..3N-1 of R, then 4N rows of A (x, y, z, low part of x), then N rows of S; chains
// [k0, k0+nk), external element (row, k) at row*pitch + (k - k0).
// A CTA owns 32 consecutive chains = G whole tiles and transposes them through shared memory, so that
// both sides of the copy move whole lines: an external row is read / written by a warp, lane = chain
// (128 contiguous bytes per request), the tiles 16 bytes per thread.  In between the 7N float rows sit
// in a staging array [row][33] (element (row, chain) in bank (row + chain) mod 32: the row accesses
// and the gathers / scatters of a tile word's four elements are both free of bank conflicts for
// N = 8, 32, 64 and two- or four-way for 16 and 128) and S as bytes [chain][8G + 4] (an odd number of words
// per chain: the row accesses, a byte per lane, and the 4-slot words of the tile side are both conflict-free).
// The import brings its rows in with 4-byte asynchronous copies (cp.async), one row per warp instruction and all
// 7N/8 rows of a warp in flight at once; the export's scattered side is its stores, which wait for nothing.
// (History, config 4, 1.96 GB: one thread per element storing straight into the tiles touched a
// 32-byte sector per word, 6.7 ms; an image of the tiles in shared memory with the external rows
// moved as 32-byte pieces, 8 chains x 4 rows per warp request, import 0.48 ms = 62 % of the copy
// bandwidth, export 0.57 ms; more of those loads in flight per thread changed nothing, whole-line
// requests through registers took the export to 0.43 ms and left the import latency-bound at 0.59;
// with the asynchronous copies it takes 0.40 ms.)
// On import the CTA also counts Z_k = number of occupied slots (they must be the leading ones).
// ---------------------------------------------------------------------------------------
constexpr int kXferPad = 33;
__host__ __device__ constexpr int xfer_smem(int N, int NP) { return 7 * N * kXferPad * 4 + 32 * (NP + 4) + 128; }

template <bool EXPORT, int G>
__global__ void __launch_bounds__(256, G <= 4 ? 6 : (G == 8 ? 3 : 1))
ssm_xfer_kernel(unsigned char *state, float *R, float *A, unsigned char *S, int N, long long k0, long long nk, long long pitch,
                int hide_low, int *bad_state)
{
    extern __shared__ __align__(16) unsigned char xs[];
    constexpr int NP = kBPL * G, cpw = 32 / G;
    constexpr int lg = G == 1 ? 0 : (G == 2 ? 1 : (G == 4 ? 2 : (G == 8 ? 3 : 4)));
    constexpr int W16 = kTileBytes / 16, WR = (kTileA - kTileR) / 16, WA = (kTileS - kTileA) / 16, WS = (kTileZ - kTileS) / 16;
    float *stg = reinterpret_cast<float *>(xs);                                  // [7N][33]: rows of R, then rows of A
    constexpr int SST = NP + 4;
    unsigned char *sS = xs + 7 * N * kXferPad * 4;                               // [32][SST]
    int *sZ = reinterpret_cast<int *>(sS + 32 * SST);                            // [32]
#ifdef SSM_CHECK
    // poisoned shared memory in the checked build (see ssm_step.cu)
    for (int i = threadIdx.x; i < xfer_smem(N, NP) / 4; i += 256) reinterpret_cast<unsigned *>(xs)[i] = 0xFFFFFFFFu;
    __syncthreads();
#endif
    const long long cb = (k0 / 32 + blockIdx.x) * 32;           // first of this CTA's 32 chains
    const long long t0 = cb / cpw, t_last = (k0 + nk - 1) / cpw;
    const int nt = (int)(t_last - t0 + 1 < (long long)G ? t_last - t0 + 1 : (long long)G);    // tiles that exist
    // a CTA whose 32 chains are all in [k0, k0 + nk) writes its tiles whole; another leaves the rest of them as it is
    const bool full = cb >= k0 && cb + 32 <= k0 + nk;
    uint4 *g4 = reinterpret_cast<uint4 *>(state + t0 * kTileBytes);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long kl = cb + lane - k0;                        // this lane's chain in the external rows
    const bool in = kl >= 0 && kl < nk;
    auto chain_in = [&](int c32) -> bool { const long long k = cb + c32 - k0; return k >= 0 && k < nk; };

    // word wi of tile T: whose chain(s) it belongs to and where its elements sit in the staging arrays
    // R word: float4 v of lane ln = cw G + g; element e is coordinate f % 3 of bead 8g + f / 3, f = 4v + e
    // A word: anchor (cw, slot j), rows 3N + c N + j;  S word: 16 bytes of [cw][slot];  Z word: 4 chains
    // The 16-byte words of a tile's R and A parts are moved in units of 32 (one per lane), 14 per tile: unit 0..5 =
    // float4 v of every lane of the step kernel (lane cw G + g: element e is coordinate f % 3 of bead 8g + f / 3,
    // f = 4v + e), unit 6..13 = 32 consecutive anchors (chain cw, slot j; rows 3N + c N + j).  Which unit a warp is at
    // is the same for its lanes, so the index arithmetic runs on the uniform path and a lane adds its own part.
    constexpr int LNP = lg + 3;
    const int cwl = lane >> lg, gl = lane & (G - 1);
    if (EXPORT) {
        // ---- tiles -> staging (16 bytes per thread, coalesced), then staging -> rows
        // (two units per turn, both loads ahead of the stores: the loop waits for its loads)
        for (int u0 = warp; u0 < nt * 14; u0 += 16) {
            uint4 t[2];
            int ai[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int u = u0 + 8 * h, T = u / 14, uu = u - 14 * T;
                ai[h] = (uu - 6) * 32 + lane;
                if (u < nt * 14) t[h] = g4[T * W16 + (uu < 6 ? uu * 32 + lane : WR + ai[h])];
            }
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int u = u0 + 8 * h, T = u / 14, uu = u - 14 * T;
                if (u >= nt * 14) continue;
                const unsigned x[4] = {t[h].x, t[h].y, t[h].z, (uu >= 6 && hide_low) ? 0u : t[h].w};
                if (uu < 6) {
                    float *sp = stg + (kBPL * gl) * kXferPad + T * cpw + cwl;
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int f = 4 * uu + e, q = f / 3, c = f - 3 * q;
                        if (kBPL * gl + q < N) sp[(c * N + q) * kXferPad] = __uint_as_float(x[e]);
                    }
                } else {
                    const int cw = ai[h] >> LNP, j = ai[h] & (NP - 1);
                    float *sp = stg + (3 * N + j) * kXferPad + T * cpw + cw;
                    if (j < N) {
#pragma unroll
                        for (int c = 0; c < 4; ++c) sp[c * N * kXferPad] = __uint_as_float(x[c]);
                    }
                }
            }
        }
        for (int i = threadIdx.x; i < nt * WS; i += 256) {
            const int T = i / WS, wi = i - T * WS;
            const uint4 t = g4[T * W16 + WR + WA + wi];
            const unsigned x[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int bi = wi * 16 + 4 * e, cw = bi >> LNP, j = bi & (NP - 1);
                *reinterpret_cast<unsigned *>(sS + (T * cpw + cw) * SST + j) = x[e];
            }
        }
        __syncthreads();
        if (in) {
            {
                float *row = R + (long long)warp * pitch + kl;
                const float *sp = stg + warp * kXferPad + lane;
                for (int r = warp; r < 3 * N; r += 8, row += 8 * pitch, sp += 8 * kXferPad) *row = *sp;
            }
            {
                float *row = A + (long long)warp * pitch + kl;
                const float *sp = stg + (3 * N + warp) * kXferPad + lane;
                for (int r = warp; r < 4 * N; r += 8, row += 8 * pitch, sp += 8 * kXferPad) *row = *sp;
            }
            unsigned char *row = S + (long long)warp * pitch + kl;
            for (int j = warp; j < N; j += 8, row += 8 * pitch) *row = sS[lane * SST + j];
        }
        return;
    }

    // ---- import: rows -> staging, asynchronously (a row's 128 bytes per warp instruction, no register in between, so
    // that a warp has all its 7N/8 rows in flight at once: the kernel is bound by the latency of these loads);
    // a lane whose chain is outside [k0, k0 + nk) is filled with zero (source size 0)
    // (hide_low is an export matter; the 4th row of A is taken as it comes)
    {
        const unsigned dst0 = (unsigned)__cvta_generic_to_shared(stg + lane);
        const unsigned nbytes = in ? 4u : 0u;
        const long long kls = in ? kl : 0;
        {
            const float *src = R + (long long)warp * pitch + kls;
            unsigned dst = dst0 + (unsigned)(warp * kXferPad * 4);
            for (int r = warp; r < 3 * N; r += 8, src += 8 * pitch, dst += 8 * kXferPad * 4)
                asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(nbytes) : "memory");
        }
        {
            const float *src = A + (long long)warp * pitch + kls;
            unsigned dst = dst0 + (unsigned)((3 * N + warp) * kXferPad * 4);
            for (int r = warp; r < 4 * N; r += 8, src += 8 * pitch, dst += 8 * kXferPad * 4)
                asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(nbytes) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
#pragma unroll 4
    for (int j = warp; j < NP; j += 8) sS[lane * SST + j] = in && j < N ? S[(long long)j * pitch + kl] : (unsigned char)0;
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    // Z = the leading occupied slots.  A caller's S must hold bead indices 1..N there and 0 after
    // them; anything else would send the step kernel's scatter outside the chain.  Such a chain keeps its
    // valid leading slots only, the rest is cleared, and the flag makes ssm_set_state fail.
    // Eight threads per chain, thread q looks at the slots [q NS, (q + 1) NS) of its chain.
    {
        constexpr int NS = NP >= 32 ? NP / 8 : 4, NQ = NP / NS;     // slots per thread, threads of a chain that have any
        const int c32 = threadIdx.x >> 3, q = threadIdx.x & 7;
        unsigned *sp = reinterpret_cast<unsigned *>(sS + c32 * SST) + q * (NS / 4);
        unsigned wd[NS / 4];
        int lead = 0;
        bool run = q < NQ;
#pragma unroll
        for (int i = 0; i < NS / 4; ++i) {
            wd[i] = q < NQ ? sp[i] : 0u;
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const unsigned by = (wd[i] >> (8 * e)) & 0xFFu;
                run = run && by != 0u && by <= (unsigned)N;
                lead += run ? 1 : 0;
            }
        }
        // the chain's first thread whose slots are not all occupied
        const unsigned fullmask = (__ballot_sync(0xffffffffu, run) >> (lane & 24)) & 0xFFu;
        const int qs = __ffs(~fullmask) - 1;                                  // 0..8
        const int lead_s = __shfl_sync(0xffffffffu, lead, (lane & 24) + (qs & 7));
        const int Z = qs >= NQ ? NP : qs * NS + lead_s;
        SSM_ASSERT(Z >= 0 && Z <= N);
        // whatever sits at or after slot Z is cleared
        bool bad = false;
        if (q < NQ && q >= qs) {
#pragma unroll
            for (int i = 0; i < NS / 4; ++i) {
                unsigned keep = 0u;
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    if (q * NS + 4 * i + e < Z) keep |= 0xFFu << (8 * e);
                if (wd[i] & ~keep) { bad = true; sp[i] = wd[i] & keep; }
            }
        }
        if (bad) atomicExch(bad_state, 1);
        if (q == 0) sZ[c32] = Z;
    }
    __syncthreads();
    // ---- staging -> tiles (16 bytes per thread, coalesced); beads and anchors: a word belongs to one chain
    for (int u = warp; u < nt * 14; u += 8) {
        const int T = u / 14, uu = u - 14 * T;
        unsigned x[4] = {0u, 0u, 0u, 0u};
        int c32;
        uint4 *q;
        if (uu < 6) {
            c32 = T * cpw + cwl;
            const float *sp = stg + (kBPL * gl) * kXferPad + c32;
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int f = 4 * uu + e, qd = f / 3, c = f - 3 * qd;
                if (kBPL * gl + qd < N) x[e] = __float_as_uint(sp[(c * N + qd) * kXferPad]);
            }
            q = g4 + T * W16 + uu * 32 + lane;
        } else {
            const int ai = (uu - 6) * 32 + lane, cw = ai >> LNP, j = ai & (NP - 1);
            c32 = T * cpw + cw;
            const float *sp = stg + (3 * N + j) * kXferPad + c32;
            if (j < N) {
#pragma unroll
                for (int c = 0; c < 4; ++c) x[c] = __float_as_uint(sp[c * N * kXferPad]);
            }
            q = g4 + T * W16 + WR + ai;
        }
        SSM_ASSERT(c32 < 32 && T < nt);
        if (full || chain_in(c32)) *q = make_uint4(x[0], x[1], x[2], x[3]);
    }
    // bead indices (16 slots of one chain, or of two 8-bead chains) and Z (4 chains): a word may hold chains in and
    // out of the range, so a CTA that is not whole blends with what the tile holds
    for (int i = threadIdx.x; i < nt * (W16 - WR - WA); i += 256) {
        const int T = i / (W16 - WR - WA), wi = i - T * (W16 - WR - WA);
        unsigned x[4] = {0u, 0u, 0u, 0u}, keep[4] = {0u, 0u, 0u, 0u};              // keep: bits that stay as they are
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            if (wi >= WS) {
                const int cw = (wi - WS) * 4 + e, c32 = T * cpw + cw;
                if (cw >= cpw) continue;
                if (full || chain_in(c32)) x[e] = (unsigned)sZ[c32]; else keep[e] = 0xFFFFFFFFu;
            } else {
                const int bi = wi * 16 + 4 * e, cw = bi >> LNP, j = bi & (NP - 1), c32 = T * cpw + cw;
                SSM_ASSERT(cw < cpw && j + 3 < NP);
                if (full || chain_in(c32)) x[e] = *reinterpret_cast<const unsigned *>(sS + c32 * SST + j); else keep[e] = 0xFFFFFFFFu;
            }
        }
        uint4 *q = g4 + T * W16 + WR + WA + wi;
        if (keep[0] | keep[1] | keep[2] | keep[3]) {
            const uint4 o = *q;
            x[0] |= o.x & keep[0]; x[1] |= o.y & keep[1]; x[2] |= o.z & keep[2]; x[3] |= o.w & keep[3];
        }
        *q = make_uint4(x[0], x[1], x[2], x[3]);
    }
}

template <bool EXPORT, int G>
static cudaError_t launch_xfer_g(unsigned grid, cudaStream_t st, unsigned char *state, float *R, float *A, unsigned char *S, int N,
                                 long long k0, long long nk, long long pitch, int hide_low, int *bad_state)
{
    // the attribute belongs to the (function, device) pair: remember per device where it has been set
    static std::atomic<unsigned long long> configured{0ull};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev >= 64 || !((configured.load(std::memory_order_relaxed) >> dev) & 1ull)) {
        if ((e = cudaFuncSetAttribute(ssm_xfer_kernel<EXPORT, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, xfer_smem(kBPL * G, kBPL * G))) != cudaSuccess) return e;
        if (dev < 64) configured.fetch_or(1ull << dev, std::memory_order_relaxed);
    }
    ssm_xfer_kernel<EXPORT, G><<<grid, 256, xfer_smem(N, kBPL * G), st>>>(state, R, A, S, N, k0, nk, pitch, hide_low, bad_state);
    return cudaGetLastError();
}

cudaError_t launch_xfer(bool do_export, unsigned char *state, float *R, float *A, unsigned char *S, int N,
                        long long k0, long long nk, long long pitch, int hide_low, int *bad_state, cudaStream_t st)
{
    if (nk <= 0) return cudaSuccess;
    const unsigned grid = (unsigned)((k0 + nk - 1) / 32 - k0 / 32 + 1);
#define SSM_XFER(G) (do_export ? launch_xfer_g<true, G>(grid, st, state, R, A, S, N, k0, nk, pitch, hide_low, bad_state) \
                               : launch_xfer_g<false, G>(grid, st, state, R, A, S, N, k0, nk, pitch, 0, bad_state))
    switch (padded_beads(N)) {
        case 8: return SSM_XFER(1);
        case 16: return SSM_XFER(2);
        case 32: return SSM_XFER(4);
        case 64: return SSM_XFER(8);
        case 128: return SSM_XFER(16);
    }
#undef SSM_XFER
    return cudaErrorInvalidValue;
}

// ---------------------------------------------------------------------------------------
// Per-chain stress of the current state (eqs 16 and 76): out[t][k], t = 0..11.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) ssm_chain_stress_kernel(const unsigned char *state, float *out, int N,
                                                               long long M, float cs)
{
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= M) return;
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
    for (int t = 0; t < 6; ++t) { out[(long long)t * M + k] = sg[t]; out[(long long)(6 + t) * M + k] = sv[t]; }
}

cudaError_t launch_chain_stress(const unsigned char *state, float *out, int N, long long M, float cs, cudaStream_t st)
{
    ssm_chain_stress_kernel<<<(unsigned)((M + 127) / 128), 128, 0, st>>>(state, out, N, M, cs);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// Clear the fourth word of every anchor (the low part(s) of the compensated advection): run when
// the flow changes between simple shear and a general tensor, whose encodings of that word differ.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) ssm_clear_low_kernel(unsigned char *state, long long n_tiles)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;      // (tile, slot of the warp)
    if (i >= n_tiles * 256) return;
    reinterpret_cast<float4 *>(state + (i >> 8) * kTileBytes + kTileA)[i & 255].w = 0.0f;
}

cudaError_t launch_clear_low(unsigned char *state, long long n_tiles, cudaStream_t st)
{
    ssm_clear_low_kernel<<<(unsigned)((n_tiles * 256 + 255) / 256), 256, 0, st>>>(state, n_tiles);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// Stress of the current state per GROUP of chains_per_group consecutive local chains (eqs 16, 76
// averaged by eq 54 over each group) and the groups' slip-spring counts: what a flow solver that
// gives every group its own velocity gradient reads back.  One thread per chain;
// out[group][13] int64 fixed point 2^-kStressShift: sigma[6], sigma_v[6], Z.  Integer sums, so the
// result does not depend on the order of the atomics.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) ssm_group_stress_kernel(const unsigned char *state, long long *out, int N,
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
        if (one_group) {
            for (int o = 16; o >= 1; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
            if ((threadIdx.x & 31) == 0) atomicAdd(reinterpret_cast<unsigned long long *>(out + group * 13 + t), (unsigned long long)v);
        } else if (valid) atomicAdd(reinterpret_cast<unsigned long long *>(out + group * 13 + t), (unsigned long long)v);
    }
}

// ---------------------------------------------------------------------------------------
// Translate every chain so that its first bead sits at the origin (beads and anchors alike).  Forces,
// hop probabilities and both stresses depend on differences R_i - R_j and R_S - A only, so nothing
// observable changes; under a flow with a stretching direction the absolute coordinates (the chain's
// centre drifts as exp(kappa t)) would otherwise use up the fp32 mantissa.  The anchors' low words
// are cleared (their unit is tied to the coordinate's exponent).
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) ssm_recenter_kernel(unsigned char *state, int N, long long M)
{
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= M) return;
    const int NP = padded_beads(N);
    float o[3];
    for (int c = 0; c < 3; ++c) o[c] = *reinterpret_cast<const float *>(state + off_R(k, NP, 0, c));
    for (int i = 0; i < N; ++i)
        for (int c = 0; c < 3; ++c) *reinterpret_cast<float *>(state + off_R(k, NP, i, c)) -= o[c];
    const int Z = *reinterpret_cast<const int *>(state + off_Z(k, NP));
    for (int j = 0; j < Z; ++j) {
        for (int c = 0; c < 3; ++c) *reinterpret_cast<float *>(state + off_A(k, NP, j, c)) -= o[c];
        *reinterpret_cast<float *>(state + off_A(k, NP, j, 3)) = 0.0f;
    }
}

cudaError_t launch_recenter(unsigned char *state, int N, long long M, cudaStream_t st)
{
    ssm_recenter_kernel<<<(unsigned)((M + 127) / 128), 128, 0, st>>>(state, N, M);
    return cudaGetLastError();
}

// dt kappa as the step kernel reads it (float) from a device table of tensors in double
__global__ void __launch_bounds__(256) ssm_kappa_kernel(const double *kappa, float *out, long long n, double dt)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = (float)(kappa[i] * dt);
}

cudaError_t launch_kappa(const double *d_kappa, float *out, long long n, double dt, cudaStream_t st)
{
    ssm_kappa_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_kappa, out, n, dt);
    return cudaGetLastError();
}

// group means from the fixed-point sums of ssm_group_stress_kernel: out[g][t] = sum / (2^kStressShift * chains in g)
__global__ void __launch_bounds__(256) ssm_group_mean_kernel(const long long *sums, double *out, long long n_groups,
                                                             long long M, long long cpg)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_groups * 13) return;
    const long long g = i / 13, n = (g + 1) * cpg <= M ? cpg : M - g * cpg;
    out[i] = (double)sums[i] / ((double)(1 << kStressShift) * (double)n);
}

cudaError_t launch_group_mean(const long long *sums, double *out, long long n_groups, long long M, long long cpg,
                              cudaStream_t st)
{
    ssm_group_mean_kernel<<<(unsigned)((n_groups * 13 + 255) / 256), 256, 0, st>>>(sums, out, n_groups, M, cpg);
    return cudaGetLastError();
}

cudaError_t launch_group_stress(const unsigned char *state, long long *out, int N, long long M, long long cpg, float cs,
                                cudaStream_t st)
{
    ssm_group_stress_kernel<<<(unsigned)((M + 127) / 128), 128, 0, st>>>(state, out, N, M, cpg, cs);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// Calibration of the Box-Muller amplitude.  The noise of eqs 44, 46 is r cos(theta), r sin(theta)
// with r = sqrt.approx(bm lg2.approx(u_a)) on the 2^16 codes of u_a and sin / cos.approx on the 2^16 angles (reading
// R24): a finite table, so the variance this GPU really delivers for a given fp32 constant bm is a finite sum that can be
// formed exactly.  The special-function unit's errors are not zero-mean (about 1.7e-7 of the variance), and bm itself is
// rounded to fp32: a SYSTEMATIC relative error of the variance, which becomes 2 eps (N - 1) of the diagonal stress
// 3 sum b_a^2 - N.  This kernel returns, for n_cand neighbouring floats bm_c = bm0 moved by c - n_cand/2 ulps,
//   out[c] = sum over the 65536 codes of r(bm_c)^2,   out[n_cand] = sum cos^2,   out[n_cand + 1] = sum sin^2   (fp64),
// and the host picks the candidate whose variance is closest to the exact sigma^2 mean(-2 ln u_a) / 2 (ssm_api.cu).
// One CTA of 1024 threads; runs once per (device, constant), not per step.
// ---------------------------------------------------------------------------------------
constexpr int kCalibMaxCand = 17;
__global__ void __launch_bounds__(1024) ssm_bm_calib_kernel(float bm0, int n_cand, double *out)
{
    __shared__ double red[32][kCalibMaxCand + 2];
    double acc[kCalibMaxCand + 2];
#pragma unroll
    for (int i = 0; i < kCalibMaxCand + 2; ++i) acc[i] = 0.0;
    for (uint32_t k = threadIdx.x; k < 65536u; k += 1024u) {
        const uint32_t w = k | (k << 16);                  // the same code in both halves: radius from the low, angle from the high
#pragma unroll
        for (int c = 0; c < kCalibMaxCand; ++c)
            if (c < n_cand) {
                const BoxMuller bm(__int_as_float(__float_as_int(bm0) + (c - n_cand / 2)));
                const double r = (double)bm.radius(w);
                acc[c] += r * r;
            }
        const float th = BoxMuller::angle(w);
        const double co = (double)__cosf(th), si = (double)__sinf(th);
        acc[kCalibMaxCand] += co * co; acc[kCalibMaxCand + 1] += si * si;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int i = 0; i < kCalibMaxCand + 2; ++i) {
        double v = acc[i];
        for (int o = 16; o >= 1; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp][i] = v;
    }
    __syncthreads();
    if (threadIdx.x < kCalibMaxCand + 2) {
        double v = 0.0;
        for (int wq = 0; wq < 32; ++wq) v += red[wq][threadIdx.x];
        const int i = threadIdx.x;
        if (i < n_cand) out[i] = v;
        else if (i >= kCalibMaxCand) out[n_cand + (i - kCalibMaxCand)] = v;
    }
}

cudaError_t launch_bm_calib(float bm0, int n_cand, double *d_out, cudaStream_t st)
{
    if (n_cand < 1 || n_cand > kCalibMaxCand) return cudaErrorInvalidValue;
    ssm_bm_calib_kernel<<<1, 1024, 0, st>>>(bm0, n_cand, d_out);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// Multi-tau correlator (BASELINE.json config 2).  One thread per chain.
// Level l holds the last P values of g block-averaged over 2^l samples; inserting (f, g)
// at level l adds f * g_(k entries ago) to sum[group][l][k] for k = kmin .. filled-1
// (kmin = 0 on level 0, P/2 above), then feeds the running pair; every second insertion
// pushes the pair's mean to level l+1.  Every chain receives the same number of samples,
// so ring positions, fill counts and pair parities are the same for all chains: they live
// on the host (which also keeps the product counts) and are replayed here from their
// values at the start of the launch.  Sums are int64 fixed point (2^-16) so that the
// result does not depend on the order of the atomics.
// ---------------------------------------------------------------------------------------
// One round of a warp-wide transposing sum: every lane holds 2H partial sums v[0..2H); lanes whose bit o is set
// keep the upper H and send the lower H to their partner (lane ^ o), the others the other way round; afterwards
// v[0..H) are sums over twice as many lanes.  Five rounds (H = 16, 8, 4, 2, 1 with o = 16, 8, 4, 2, 1) turn 32
// values per lane into ONE total per lane, value number = lane: 31 shuffles instead of 32 warp reductions.
template <int H>
__device__ __forceinline__ void transpose_sum_round(int (&v)[32], int o, int lane)
{
    const bool up = (lane & o) != 0;
#pragma unroll
    for (int i = 0; i < H; ++i) {
        const int send = up ? v[i] : v[i + H];
        const int keep = up ? v[i + H] : v[i];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, o);
    }
}

__global__ void __launch_bounds__(256) ssm_corr_kernel(const __grid_constant__ CorrParams C)
{
    // one thread per HISTORY k = q M + chain (component q = xy, or xy / yz / zx), Mv = n_comp M of them
    const long long k0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = k0 < C.Mv;
    const long long k = valid ? k0 : C.Mv - 1;          // idle lanes of the last warp shadow a real history and add 0
    const int L = C.L, Pb = C.Pb, lane = threadIdx.x & 31;
    // group = (global chain index / 32) % groups: the same for the whole warp when the local chain 0
    // sits on a multiple of 32 and M is one (else the per-lane path below takes over)
    const int group = (int)(((C.chain_offset + (unsigned long long)(k % C.M)) >> 5) % (unsigned)C.groups);
    const bool one_group = __all_sync(0xffffffffu, group == __shfl_sync(0xffffffffu, group, 0));
    long long *gsum = C.sum + (long long)group * L * Pb, *gsum2 = C.sum_gg + (long long)group * L * Pb;
    unsigned char pos[kCorrMaxLevels], fil[kCorrMaxLevels], par[kCorrMaxLevels];
    for (int lev = 0; lev < L; ++lev) { pos[lev] = C.pos[lev]; fil[lev] = C.filled[lev]; par[lev] = C.parity[lev]; }
    for (int s = 0; s < C.n_samples; ++s) {
        const float2 fg = C.samples[(long long)s * C.Mv + k];
        float f = fg.x, g = fg.y;
        for (int lev = 0; lev < L; ++lev) {              // (every bound in here is the same for all chains)
            const long long lm = (long long)lev * C.Mv + k;
            float *ring = C.ring + (long long)lev * Pb * C.Mv + k;
            const int p0 = pos[lev];
            SSM_ASSERT(p0 >= 0 && p0 < Pb && k >= 0 && k < C.Mv && group >= 0 && group < C.groups);
            if (valid) ring[(long long)p0 * C.Mv] = g;
            if (fil[lev] < Pb) ++fil[lev];
            const int kmin = lev == 0 ? 0 : Pb / 2, kfil = fil[lev];
            // the bins of this insertion, 16 at a time: products in fixed point 2^-16, f_new g_old for G(t)
            // (eq 43) at even places and g_new g_old for the virtual-stress share (eq 66) at odd places
            for (int q0 = kmin; q0 < kfil; q0 += 16) {
                const int nb = kfil - q0 < 16 ? kfil - q0 : 16;
                float pf[16], pg[16], big = 0.0f;
#pragma unroll
                for (int b = 0; b < 16; ++b) {
                    int idx = p0 - (q0 + b); if (idx < 0) idx += Pb;
                    const float old = (valid && b < nb) ? ring[(long long)idx * C.Mv] : 0.0f;
                    pf[b] = f * old * 65536.0f; pg[b] = g * old * 65536.0f;
                    big = fmaxf(big, fmaxf(fabsf(pf[b]), fabsf(pg[b])));
                }
                if (one_group && !__any_sync(0xffffffffu, !(big < 3.3e7f))) {
                    // every |product| < 2^25, so the sum over the warp's 32 chains fits 32 bits: one transposing
                    // sum gives lane i the warp's total of value i, and the 32 lanes add their totals at once
                    int v[32];
#pragma unroll
                    for (int b = 0; b < 16; ++b) { v[2 * b] = __float2int_rn(pf[b]); v[2 * b + 1] = __float2int_rn(pg[b]); }
                    int mine_bin, total;
                    if (nb > 8) {
                        transpose_sum_round<16>(v, 16, lane); transpose_sum_round<8>(v, 8, lane);
                        transpose_sum_round<4>(v, 4, lane); transpose_sum_round<2>(v, 2, lane);
                        transpose_sum_round<1>(v, 1, lane);
                        total = v[0]; mine_bin = lane >> 1;
                    } else {
                        // 16 values only (the upper levels): four rounds leave value number lane >> 1 in the two
                        // lanes of a pair, which share the bin's two sums between them
                        transpose_sum_round<8>(v, 16, lane); transpose_sum_round<4>(v, 8, lane);
                        transpose_sum_round<2>(v, 4, lane); transpose_sum_round<1>(v, 2, lane);
                        total = v[0] + __shfl_xor_sync(0xffffffffu, v[0], 1);
                        mine_bin = (lane >> 2) | ((lane & 1) ? 16 : 0);      // the odd lane of a pair stays idle
                    }
                    const bool gg = nb > 8 ? (lane & 1) != 0 : (lane & 2) != 0;
                    if (mine_bin < nb && total != 0)
                        atomicAdd(reinterpret_cast<unsigned long long *>((gg ? gsum2 : gsum) + lev * Pb + q0 + mine_bin),
                                  (unsigned long long)(long long)total);
                } else {
                    for (int b = 0; b < nb; ++b) {
                        float pfb = 0.f, pgb = 0.f;
#pragma unroll
                        for (int e = 0; e < 16; ++e) if (e == b) { pfb = pf[e]; pgb = pg[e]; }
                        const long long v = __float2ll_rn(pfb), v2 = __float2ll_rn(pgb);
                        const int q = q0 + b;
                        if (one_group) {
                            // exact warp sums of the 64-bit values as two 32-bit integer reductions each:
                            // v = hi 2^20 + lo, 0 <= lo < 2^20 (|v| < 2^46 keeps the sum of 32 hi's in 32 bits)
                            const int hi = __reduce_add_sync(0xffffffffu, (int)(v >> 20));
                            const int lo = __reduce_add_sync(0xffffffffu, (int)(v & 0xFFFFF));
                            const int hi2 = __reduce_add_sync(0xffffffffu, (int)(v2 >> 20));
                            const int lo2 = __reduce_add_sync(0xffffffffu, (int)(v2 & 0xFFFFF));
                            if (lane == 0) {
                                atomicAdd(reinterpret_cast<unsigned long long *>(gsum + lev * Pb + q),
                                          (unsigned long long)(((long long)hi << 20) + (long long)lo));
                                atomicAdd(reinterpret_cast<unsigned long long *>(gsum2 + lev * Pb + q),
                                          (unsigned long long)(((long long)hi2 << 20) + (long long)lo2));
                            }
                        } else if (valid) {
                            atomicAdd(reinterpret_cast<unsigned long long *>(gsum + lev * Pb + q), (unsigned long long)v);
                            atomicAdd(reinterpret_cast<unsigned long long *>(gsum2 + lev * Pb + q), (unsigned long long)v2);
                        }
                    }
                }
            }
            pos[lev] = (unsigned char)((p0 + 1) % Pb);
            if (par[lev] == 0) {
                if (valid) { C.acc_f[lm] = f; C.acc_g[lm] = g; }
                par[lev] = 1;
                break;
            }
            f = 0.5f * (C.acc_f[lm] + f); g = 0.5f * (C.acc_g[lm] + g);
            par[lev] = 0;
        }
    }
}

cudaError_t launch_corr(const CorrParams &c, cudaStream_t st)
{
    ssm_corr_kernel<<<(unsigned)((c.Mv + 255) / 256), 256, 0, st>>>(c);
    return cudaGetLastError();
}

}  // namespace ssm

namespace ssm {
// ---------------------------------------------------------------------------------------
// Issue-rate probe (DIAGNOSTIC): cycles per group of instructions per scheduler, measured
// at the step kernel's residency (4 warps per scheduler) with 4 independent chains per lane.  A group is
//   NW x [IMAD.WIDE.U32 + the LOP3 that folds its two halves]  (the Philox round's pattern),
//   NL x LOP3 (ALU pipe), NF x FFMA, NM x MUFU.EX2, NI x IMAD (low half), NY x [I2FP + F2I].
// What the step kernel's roofline needs from it: the ALU pipe takes 2 cycles per LOP3-class instruction; IMAD 2;
// the 32 x 32 -> 64-bit multiply holds the ISSUE port, not just its pipe -- FFMAs put beside it do not hide
// (group of one multiply + n FFMA = multiply + n cycles), so each one costs ~3 issue cycles beyond its own slot.
// ---------------------------------------------------------------------------------------
template <int NW, int NL, int NF, int NM, int NI, int NY>
__global__ void __launch_bounds__(512) ssm_rate_kernel(unsigned *out, int iters, unsigned seed)
{
    constexpr int ILP = 4;
    unsigned a[ILP], l[ILP][4], im[ILP][2]; float f[ILP][4], m[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) {
        a[i] = seed + threadIdx.x * 7u + i; m[i] = 0.5f + 1e-3f * threadIdx.x;
#pragma unroll
        for (int j = 0; j < 4; ++j) { l[i][j] = seed + 11u * j + i + threadIdx.x; f[i][j] = 1.0f + 1e-3f * (j + i + threadIdx.x); }
        im[i][0] = seed + threadIdx.x; im[i][1] = seed * 5u + threadIdx.x;
    }
    const long long t0 = clock64();
    for (int n = 0; n < iters; ++n) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) {
#pragma unroll
            for (int w = 0; w < NW; ++w) a[i] = __umulhi(a[i], 0xD2511F53u) ^ (a[i] * 0xD2511F53u);
#pragma unroll
            for (int j = 0; j < NL; ++j) asm volatile("lop3.b32 %0, %0, %1, 0x9E3779B9, 0x96;" : "+r"(l[i][j & 3]) : "r"(l[i][(j + 1) & 3]));
#pragma unroll
            for (int j = 0; j < NF; ++j) asm volatile("fma.rn.f32 %0, %0, %1, %1;" : "+f"(f[i][j & 3]) : "f"(f[i][(j + 1) & 3]));
#pragma unroll
            for (int j = 0; j < NM; ++j) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(m[i]));
#pragma unroll
            for (int j = 0; j < NI; ++j) asm volatile("mad.lo.u32 %0, %0, 0xCD9E8D57, %1;" : "+r"(im[i][j & 1]) : "r"(im[i][(j + 1) & 1]));
#pragma unroll
            for (int j = 0; j < NY; ++j) { float t; asm volatile("cvt.rn.f32.s32 %0, %1;" : "=f"(t) : "r"(l[i][j & 3])); asm volatile("cvt.rni.s32.f32 %0, %1;" : "=r"(l[i][j & 3]) : "f"(t)); }
        }
    }
    const long long t1 = clock64();
    unsigned r = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) {
        r += a[i] + __float_as_uint(m[i]) + im[i][0] + im[i][1];
#pragma unroll
        for (int j = 0; j < 4; ++j) r += l[i][j] + __float_as_uint(f[i][j]);
    }
    out[1 + blockIdx.x * blockDim.x + threadIdx.x] = r;
    if ((threadIdx.x & 31) == 0) atomicMax(out, (unsigned)(t1 - t0));      // the slowest warp of the grid
}

template <int NW, int NL, int NF, int NM, int NI, int NY>
static cudaError_t rate_one(unsigned *d_scratch, int blocks, cudaStream_t st, double *cycles_per_group)
{
    const int iters = 2000, ilp = 4, warps_per_smsp = 4;
    ssm_rate_kernel<NW, NL, NF, NM, NI, NY><<<blocks, 512, 0, st>>>(d_scratch, iters, 1u);      // warms the instruction cache
    cudaError_t e = cudaMemsetAsync(d_scratch, 0, sizeof(unsigned), st);
    if (e != cudaSuccess) return e;
    ssm_rate_kernel<NW, NL, NF, NM, NI, NY><<<blocks, 512, 0, st>>>(d_scratch, iters, 1u);
    unsigned cyc = 0;
    e = cudaMemcpyAsync(&cyc, d_scratch, sizeof cyc, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return e;
    *cycles_per_group = (double)cyc / ((double)iters * ilp * warps_per_smsp);
    return cudaGetLastError();
}

// out: device scratch of at least (1 + blocks * 512) words; cycles[8] = cycles per group of
// [0] FFMA, [1] LOP3, [2] IMAD, [3] IMAD.WIDE + LOP3, [4] IMAD.WIDE + LOP3 + 4 FFMA, [5] MUFU, [6] I2FP + F2I,
// [7] 2 x (IMAD.WIDE + LOP3): the instructions of one Philox round
cudaError_t measure_rates(unsigned *d_scratch, int blocks, cudaStream_t st, double cycles[8])
{
    cudaError_t e;
    if ((e = rate_one<0, 0, 1, 0, 0, 0>(d_scratch, blocks, st, cycles + 0)) != cudaSuccess) return e;
    if ((e = rate_one<0, 1, 0, 0, 0, 0>(d_scratch, blocks, st, cycles + 1)) != cudaSuccess) return e;
    if ((e = rate_one<0, 0, 0, 0, 1, 0>(d_scratch, blocks, st, cycles + 2)) != cudaSuccess) return e;
    if ((e = rate_one<1, 0, 0, 0, 0, 0>(d_scratch, blocks, st, cycles + 3)) != cudaSuccess) return e;
    if ((e = rate_one<1, 0, 4, 0, 0, 0>(d_scratch, blocks, st, cycles + 4)) != cudaSuccess) return e;
    if ((e = rate_one<0, 0, 0, 1, 0, 0>(d_scratch, blocks, st, cycles + 5)) != cudaSuccess) return e;
    if ((e = rate_one<0, 0, 0, 0, 0, 1>(d_scratch, blocks, st, cycles + 6)) != cudaSuccess) return e;
    return rate_one<2, 0, 0, 0, 0, 0>(d_scratch, blocks, st, cycles + 7);
}
}  // namespace ssm
