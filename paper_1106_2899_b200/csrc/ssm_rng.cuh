// ssm_rng.cuh -- counter-based random numbers of the CUDA path (device only).
//
// The paper draws w_i with "the linear congruential method and the Box-Muller transform"
// (section 3.1).  BASELINE.json's north_star replaces the LCG by
// Philox4x32-10 keyed by (seed, chain, item, step); the stream layout is DESIGN.md
// section 4 ("RNG contract").  This file is the GPU's own statement of it; it shares no
// code with oracle/.
#pragma once
#include <cstdint>

namespace ssm {

// stream domains
enum : uint32_t {
    DOM_NOISE = 0,        // per step: normal m = 3*bead + axis, call m>>3, normal m&7
    DOM_SLOT = 1,         // per step: call j>>1, words 2(j&1), 2(j&1)+1 = u_hop, u_end of slip-spring j
    DOM_ATTEMPT = 2,      // per step: call k>>3, half k&1 of word (k&7)>>1 = high 16 bits of the 23-bit code of attempt k
    DOM_ANCHOR = 3,       // per step: call k, normals 0..2 (words 0, 1) = anchor offset of attempt k,
                          //           top 7 bits of word 2 = low 7 bits of its 23-bit code
    DOM_INIT_BOND = 4,    // step 0: normal m = 3*bond + axis
    DOM_INIT_Z = 5,       // step 0, call 0, word 0 -> Z
    DOM_INIT_SLOT = 6,    // step 0, call j, word 0 -> S_j
    DOM_INIT_ANCHOR = 7   // step 0, call j, normals 0..2 -> anchor offset
};

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): ten rounds of
//   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
// the key bumped by the Weyl constants between rounds.  RK holds the 20 round keys
// (k0 + r W0, k1 + r W1): the host computes them once so that the kernel reads them from
// the constant bank instead of spending 20 additions per call.
struct RoundKeys { const unsigned *rk; };

__host__ __device__ inline void philox_round_keys(uint32_t k0, uint32_t k1, unsigned (&rk)[20])
{
    for (int r = 0; r < 10; ++r) { rk[2 * r] = k0 + (uint32_t)r * 0x9E3779B9u; rk[2 * r + 1] = k1 + (uint32_t)r * 0xBB67AE85u; }
}

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              const unsigned (&rk)[20], uint32_t (&out)[4])
{
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)M0 * c0;
        const uint64_t p1 = (uint64_t)M1 * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk[2 * r];
        c2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk[2 * r + 1];
        c1 = (uint32_t)p1; c3 = (uint32_t)p0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// counter = (step low 32, domain<<28 | step bits 32..59, global chain index, item)
//
// The first counter word (the step) is the same for every call of a time step, so what the
// first round makes of it is formed ONCE per step: M0 * step gives hi ^ k1 (xored with the
// item in round 1) and lo ^ (k1 + W1) (xored with a product in round 2).  A call then spends
// one wide multiply in round 1 instead of two, and the two xors that would take two uniform
// operands take one.  The result is Philox4x32-10 of the counter above, bit for bit.
struct StreamKey {
    uint32_t c1hi;          // step bits 32..59
    uint32_t a1;            // hi(M0 * step low 32) ^ rk[1]
    uint32_t b3;            // lo(M0 * step low 32) ^ rk[3]
};
__device__ __forceinline__ StreamKey make_stream(unsigned long long step, const unsigned (&rk)[20])
{
    const uint64_t p0 = (uint64_t)0xD2511F53u * (uint32_t)step;
    StreamKey s;
    s.c1hi = (uint32_t)(step >> 32) & 0x0FFFFFFFu;
    s.a1 = (uint32_t)(p0 >> 32) ^ rk[1];
    s.b3 = (uint32_t)p0 ^ rk[3];
    return s;
}
// The round keys of rounds 2..10 come from a copy in SHARED memory when the caller has one
// (rk_sm, 16-byte aligned, 20 words): five 16-byte broadcast loads put them straight into
// registers.  Read from the kernel parameters they arrive in uniform registers, and ptxas then
// spends a register move per key and call on them (measured: 18 moves per call in the slot pass).
template <bool SM = false>
__device__ __forceinline__ void stream_call(const StreamKey& s, const unsigned (&rk)[20], uint32_t domain,
                                            uint32_t chain, uint32_t item, uint32_t (&w)[4],
                                            const uint4 *rk_sm = nullptr)
{
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    unsigned k[20];
    if (SM) {
#pragma unroll
        for (int i = 0; i < 5; ++i) { const uint4 t = rk_sm[i]; k[4 * i] = t.x; k[4 * i + 1] = t.y; k[4 * i + 2] = t.z; k[4 * i + 3] = t.w; }
    } else {
#pragma unroll
        for (int i = 0; i < 20; ++i) k[i] = rk[i];
    }
    // round 1 on (step, domain | step hi, chain, item)
    const uint64_t q1 = (uint64_t)M1 * chain;
    uint32_t c0 = (uint32_t)(q1 >> 32) ^ (((domain << 28) | s.c1hi) ^ rk[0]);
    uint32_t c1 = (uint32_t)q1;
    uint32_t c2 = s.a1 ^ item;
    // round 2: its c3 is lo(M0 * step), already folded with rk[3] into b3
    const uint64_t p0 = (uint64_t)M0 * c0;
    const uint64_t p1 = (uint64_t)M1 * c2;
    c0 = (uint32_t)(p1 >> 32) ^ c1 ^ k[2];
    c2 = (uint32_t)(p0 >> 32) ^ s.b3;
    c1 = (uint32_t)p1;
    uint32_t c3 = (uint32_t)p0;
#pragma unroll
    for (int r = 2; r < 10; ++r) {
        const uint64_t t0 = (uint64_t)M0 * c0;
        const uint64_t t1 = (uint64_t)M1 * c2;
        c0 = (uint32_t)(t1 >> 32) ^ c1 ^ k[2 * r];
        c2 = (uint32_t)(t0 >> 32) ^ c3 ^ k[2 * r + 1];
        c1 = (uint32_t)t1; c3 = (uint32_t)t0;
    }
    w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
}

// Rounds 1 and 2 of a call depend on the step and the item only through a1 ^ item and b3: what they make of
// (domain | step bits 32..59, chain) -- c1 = lo(M1 chain) and the product M0 * [hi(M1 chain) ^ (domain | step hi) ^ k0]
// of round 2 -- is the same for every call of a (chain, domain) during a launch (the host never lets a launch cross a
// multiple of 2^32 steps).  stream_prefix() forms that part once per tile; stream_call_pre() is stream_call() with
// it: two wide multiplies and an xor fewer per call, bit for bit the same words.
__device__ __forceinline__ uint4 stream_prefix(const StreamKey& s, const unsigned (&rk)[20], uint32_t domain, uint32_t chain)
{
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint64_t q1 = (uint64_t)M1 * chain;
    const uint32_t c0 = (uint32_t)(q1 >> 32) ^ (((domain << 28) | s.c1hi) ^ rk[0]);
    const uint64_t p0 = (uint64_t)M0 * c0;
    return make_uint4((uint32_t)q1, (uint32_t)(p0 >> 32), (uint32_t)p0, 0u);
}
__device__ __forceinline__ void stream_call_pre(const StreamKey& s, const uint4 pre, uint32_t item, uint32_t (&w)[4],
                                                const uint4 *rk_sm)
{
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    unsigned k[20];
#pragma unroll
    for (int i = 0; i < 5; ++i) { const uint4 t = rk_sm[i]; k[4 * i] = t.x; k[4 * i + 1] = t.y; k[4 * i + 2] = t.z; k[4 * i + 3] = t.w; }
    const uint64_t p1 = (uint64_t)M1 * (s.a1 ^ item);
    uint32_t c0 = (uint32_t)(p1 >> 32) ^ pre.x ^ k[2];
    uint32_t c2 = pre.y ^ s.b3;
    uint32_t c1 = (uint32_t)p1;
    uint32_t c3 = pre.z;
#pragma unroll
    for (int r = 2; r < 10; ++r) {
        const uint64_t t0 = (uint64_t)M0 * c0;
        const uint64_t t1 = (uint64_t)M1 * c2;
        c0 = (uint32_t)(t1 >> 32) ^ c1 ^ k[2 * r];
        c2 = (uint32_t)(t0 >> 32) ^ c3 ^ k[2 * r + 1];
        c1 = (uint32_t)t1; c3 = (uint32_t)t0;
    }
    w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
}

// 23-bit code k = w >> 9 and the uniform u = (k + 1/2) 2^-23 in (0,1); exact in fp32:
// [1 + k 2^-23] - [1 - 2^-24].
__device__ __forceinline__ uint32_t code23(uint32_t w) { return w >> 9; }
__device__ __forceinline__ float u23(uint32_t w)
{
    return __uint_as_float(0x3F800000u | (w >> 9)) - 0.99999994f;
}

__device__ __forceinline__ float mufu_sqrt(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float mufu_lg2(float x)
{
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Box-Muller on ONE Philox word (reading R24): the low and the high half
// are 16-bit codes ka, kb; u_a = (ka + 1/2) 2^-16, theta = 2 pi ((kb + 1/2) 2^-16 - 1/2);
// (z0, z1) = (r cos theta, r sin theta) with r = sigma sqrt(-2 ln u_a) are two N(0, sigma^2)
// numbers, so a Philox call yields EIGHT normals.  bm = -2 ln2 sigma^2, so that
// r^2 = bm log2(u_a).  The special-function unit evaluates log2, sqrt, sin and cos (absolute
// error <= 2^-21.4 each in the ranges used here; log2 is taken of
// u_a in (0,1) itself so that it keeps its relative accuracy where u_a -> 1).  Both codes are
// turned into floats exactly with one byte permute each: the bytes of the half word under
// the exponent of 2^23 give the float 2^23 + k, and (2^23 + ka) 2^-16 - (128 - 2^-17) = u_a
// is one exact fused multiply-add.
struct BoxMuller {
    float bm;            // -2 ln2 sigma^2
    __device__ __forceinline__ explicit BoxMuller(float b) : bm(b) {}
    // radius from the low half word, angle from the high one (also called one by one by the calibration kernel of
    // ssm_aux.cu, which sums r^2, cos^2 and sin^2 over all 2^16 codes with exactly these instructions)
    __device__ __forceinline__ float radius(uint32_t w) const
    {
        const float ua = fmaf(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7610)), 1.52587890625e-05f, -127.99999237060547f);
        return mufu_sqrt(bm * mufu_lg2(ua));
    }
    static __device__ __forceinline__ float angle(uint32_t w)
    {
        const float kb = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7632)) - 8421376.0f;   // kb - 2^15
        return fmaf(kb, 9.5873799e-05f, 4.7936899e-05f);                 // 2 pi 2^-16 (kb - 2^15) + pi 2^-16
    }
    __device__ __forceinline__ void operator()(uint32_t w, float& z0, float& z1) const
    {
        const float th = angle(w);
        const float r = radius(w);
        z0 = r * __cosf(th); z1 = r * __sinf(th);
    }
};

// the eight normals of one call: (2e, 2e+1) from word e
template <bool SM = false>
__device__ __forceinline__ void normal_call(const StreamKey& s, const unsigned (&rk)[20], uint32_t domain,
                                            uint32_t chain, uint32_t call, const BoxMuller& bm, float (&z)[8],
                                            const uint4 *rk_sm = nullptr)
{
    uint32_t w[4];
    stream_call<SM>(s, rk, domain, chain, call, w, rk_sm);
#pragma unroll
    for (int e = 0; e < 4; ++e) bm(w[e], z[2 * e], z[2 * e + 1]);
}

// normals 0..2 of a call (anchor offsets, eqs 15 and 52): words 0 and 1 only
__device__ __forceinline__ void anchor_normals(const StreamKey& s, const unsigned (&rk)[20], uint32_t domain,
                                               uint32_t chain, uint32_t call, const BoxMuller& bm, float (&z)[3])
{
    uint32_t w[4];
    stream_call(s, rk, domain, chain, call, w);
    float unused;
    bm(w[0], z[0], z[1]);
    bm(w[1], z[2], unused);
}

}  // namespace ssm
