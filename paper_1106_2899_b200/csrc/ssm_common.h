// ssm_common.h -- internal layout and launch-parameter structs of libssm (host + device).
//
// Mapping: a chain of N = 4G beads is owned by G consecutive lanes of
// one warp (G = 2, 4, 8, 16, 32), 4 consecutive beads per lane, so a warp owns CPW = 32/G
// chains and never talks to another warp.  The unit of state in HBM is therefore the
// "warp tile": the register / shared-memory image of one warp's chains, stored so that a
// warp loads and stores it with fully coalesced 16-byte accesses:
//
//   bytes [   0,1536)  R image : 3 x float4 per lane, element [v][lane], float f = 4v+e of
//                                lane = coordinate (f%3) of the lane's bead f/3
//   bytes [1536,3072)  A image : [chain in warp][slot 0..zmax-1][3] float   (zmax = N)
//   bytes [3072,3200)  S image : [chain in warp][slot] uint8, 0 = empty, 1..N
//   bytes [3200,3264)  Z       : [chain in warp] int32 (16 entries, CPW used)
//   bytes [3264,3328)  pad
#pragma once
#include <cstdint>

namespace ssm {

constexpr int kTileBytes = 3328;
constexpr int kTileR = 0, kTileA = 1536, kTileS = 3072, kTileZ = 3200;
constexpr int kWarpsPerBlock = 8;
constexpr int kBlockThreads = 32 * kWarpsPerBlock;
constexpr int kMaxFuse = 32;                 // time steps fused per launch (stress accumulators in smem)
constexpr int kFxShift = 26;                 // slip-spring displacement fixed point: 2^-26 b
constexpr int kStressShift = 24;             // ensemble stress fixed point: 2^-24 kT

// per-warp shared memory of the step kernel
constexpr int kSmRm = 0;        // float[384]  bead positions mirror [chain][bead][3]
constexpr int kSmFx = 1536;     // int  [384]  fixed-point slip-spring displacement per bead coordinate
constexpr int kSmA = 3072;      // float[384]  anchors [chain][slot][3]
constexpr int kSmS = 4608;      // uint8[128]  bead index per slot
constexpr int kSmZ = 4736;      // int  [16]   Z per chain
constexpr int kSmAtt = 4800;    // uint8[128]  result of construction attempt k (0, 1 or N)
constexpr int kSmWarp = 4928;
constexpr int kSmAcc = kWarpsPerBlock * kSmWarp;                          // int64 [8][kMaxFuse][12]
constexpr int kSmStep = kSmAcc + kWarpsPerBlock * kMaxFuse * 12 * 8;      // 63,744 B + 0

struct StepParams {
    unsigned char *state;             // warp tiles
    long long     *stress;            // [capacity][12] int64 fixed-point sums; slot of this launch's first record
    float2        *samples;           // [n_sample_steps of this launch][M] (f, g) per chain, or null
    long long      n_chains;          // M (chains >= M in the last tile are padding)
    unsigned long long chain_offset;  // global index of local chain 0
    unsigned long long step0;         // global index of the first step of this launch
    int            n_tiles;
    int            n_fuse;            // steps in this launch (<= kMaxFuse)
    int            stress_every;      // 0 = never
    int            sample_every;      // 0 = never
    unsigned       key0, key1;        // Philox key
    int            springs_on;
    float dt3;        // 3 dt                 (Rouse spring constant 3kT/b^2, eq 1)
    float sq2dt;      // sqrt(2 dt)           (eq 44)
    float gdt;        // shear_rate * dt      (eq 44, 45 with kappa_xy of eq 60)
    float fx_scale;   // dt * (3/N_s) * 2^kFxShift
    float q2l;        // 2 * (3/(4 N_s)) * log2(e): exponent scale of 1 - tanh(x) = 2/(1+e^{2x})
    float h2;         // 2 dt/zeta_s
    float cs;         // 3/N_s                (eq 76)
    float sq_ns3;     // sqrt(N_s/3)          (eq 52)
    unsigned t_destroy;               // T(min{dt/zeta_s, 1})                 (eq 53)
    unsigned t_c1[129], t_c2[129];    // T(p_c(K)), T(2 p_c(K)), K = 1..128   (eqs 50, 51)
};

struct InitParams {
    unsigned char *state;
    long long      n_chains_padded;   // n_tiles * CPW
    unsigned long long chain_offset;
    unsigned       key0, key1;
    int            n_beads;
    int            springs_on;
    float          sq13;              // sqrt(1/3)   (eq 6)
    float          sq_ns3;            // sqrt(N_s/3) (eq 15)
    unsigned       t_cdf[128];        // T(P(Z <= z)), z = 0..zmax-1  (eq 12)
};

constexpr int kCorrMaxLevels = 32;
struct CorrParams {
    const float2 *samples;     // [n_samples][M] (f, g) = (sigma_xy, sigma_xy + sigma^(v)_xy)
    float *ring;               // [L][P][M] block-averaged g history
    float *acc_f, *acc_g;      // [L][M] first element of the pending pair
    long long *sum;            // [groups][L][P] int64 fixed point (2^-16)
    long long M;
    unsigned long long chain_offset;
    int n_samples, L, Pb, groups;
    unsigned char pos[kCorrMaxLevels], filled[kCorrMaxLevels], parity[kCorrMaxLevels];   // at launch start
};

// address of bead coordinate / slot entry inside the tiled state (host and device)
__host__ __device__ inline long long tile_of(long long chain, int n_beads) { return chain / (128 / n_beads); }
__host__ __device__ inline long long off_R(long long chain, int n_beads, int bead, int c)
{
    const int G = n_beads / 4, cpw = 32 / G;
    const long long tile = chain / cpw; const int cw = (int)(chain % cpw);
    const int lane = cw * G + bead / 4, f = (bead % 4) * 3 + c;
    return tile * kTileBytes + kTileR + (((f >> 2) * 32 + lane) * 4 + (f & 3)) * 4;
}
__host__ __device__ inline long long off_A(long long chain, int n_beads, int slot, int c)
{
    const int cpw = 128 / n_beads;
    return (chain / cpw) * kTileBytes + kTileA + (((int)(chain % cpw) * n_beads + slot) * 3 + c) * 4;
}
__host__ __device__ inline long long off_S(long long chain, int n_beads, int slot)
{
    const int cpw = 128 / n_beads;
    return (chain / cpw) * kTileBytes + kTileS + (int)(chain % cpw) * n_beads + slot;
}
__host__ __device__ inline long long off_Z(long long chain, int n_beads)
{
    const int cpw = 128 / n_beads;
    return (chain / cpw) * kTileBytes + kTileZ + (int)(chain % cpw) * 4;
}

}  // namespace ssm
