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
    DOM_NOISE = 0,        // per step: normal m = 3*bead + axis, call m>>2, normal m&3
    DOM_SLOT = 1,         // per step: call j>>1, words 2(j&1), 2(j&1)+1 = u_hop, u_end of slip-spring j
    DOM_ATTEMPT = 2,      // per step: call k>>2, word k&3 = uniform of construction attempt k
    DOM_ANCHOR = 3,       // per step: call k, normals 0..2 = anchor offset of attempt k
    DOM_INIT_BOND = 4,    // step 0: normal m = 3*bond + axis
    DOM_INIT_Z = 5,       // step 0, call 0, word 0 -> Z
    DOM_INIT_SLOT = 6,    // step 0, call j, word 0 -> S_j
    DOM_INIT_ANCHOR = 7   // step 0, call j, normals 0..2 -> anchor offset
};

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): ten rounds of
//   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
// the key bumped by the Weyl constants between rounds.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t (&out)[4])
{
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)M0 * c0;
        const uint64_t p1 = (uint64_t)M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ (k0 + (uint32_t)r * W0);
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ (k1 + (uint32_t)r * W1);
        c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// counter = (step low 32, domain<<28 | step bits 32..59, global chain index, item)
struct StreamKey {
    uint32_t k0, k1;        // seed low / high
    uint32_t c0, c1hi;      // step low 32 bits, step bits 32..59
};
__device__ __forceinline__ StreamKey make_stream(uint32_t k0, uint32_t k1, unsigned long long step)
{
    StreamKey s; s.k0 = k0; s.k1 = k1; s.c0 = (uint32_t)step;
    s.c1hi = (uint32_t)(step >> 32) & 0x0FFFFFFFu;
    return s;
}
__device__ __forceinline__ void stream_call(const StreamKey& s, uint32_t domain, uint32_t chain,
                                            uint32_t item, uint32_t (&w)[4])
{
    philox4x32_10(s.c0, (domain << 28) | s.c1hi, chain, item, s.k0, s.k1, w);
}

// 23-bit code k = w >> 9 and the uniform u = (k + 1/2) 2^-23 in (0,1); exact in fp32:
// [1 + k 2^-23] - [1 - 2^-24].
__device__ __forceinline__ uint32_t code23(uint32_t w) { return w >> 9; }
__device__ __forceinline__ float u23(uint32_t w)
{
    return __uint_as_float(0x3F800000u | (w >> 9)) - 0.99999994f;
}

// Box-Muller: r = sqrt(-2 ln u_a), theta = 2 pi (u_b - 1/2) = pi t with
// t = 2 u_b - 1 = (2k+1) 2^-23 - 1 formed exactly; (z0, z1) = (r cos theta, r sin theta).
__device__ __forceinline__ void box_muller(uint32_t wa, uint32_t wb, float& z0, float& z1)
{
    const float ua = u23(wa);
    const float x = __uint_as_float(0x3F800000u | (wb >> 9)) - 1.5f;   // k 2^-23 - 1/2, exact
    const float t = fmaf(2.0f, x, 1.1920929e-07f);                     // + 2^-23, exact
    const float r = sqrtf(-2.0f * logf(ua));
    float sn, cs;
    sincospif(t, &sn, &cs);
    z0 = r * cs; z1 = r * sn;
}

// the four normals of one call: (0,1) from words (0,1), (2,3) from words (2,3)
__device__ __forceinline__ void normal_call(const StreamKey& s, uint32_t domain, uint32_t chain,
                                            uint32_t call, float (&z)[4])
{
    uint32_t w[4];
    stream_call(s, domain, chain, call, w);
    box_muller(w[0], w[1], z[0], z[1]);
    box_muller(w[2], w[3], z[2], z[3]);
}

}  // namespace ssm
