// ssm_common.h -- internal layout and launch-parameter structs of libssm (host + device).
//
// Mapping: a chain of N beads is owned by G consecutive lanes of one warp,
// G = 1, 2, 4, 8, 16 the smallest with 8G >= N, 8 consecutive beads per lane, so a warp owns
// CPW = 32/G chains (256 bead places, up to 256 slip-spring slots) and never talks to another
// warp.  When N < 8G (the paper's N = 10, 20, 40, 80) the places N..8G-1 of a chain are padding:
// no bond reaches them, no slip-spring sits on them, they are kept at the origin.  Every
// "n_beads" argument of the layout helpers below is the PADDED count 8G.
// The unit of state in HBM is the "warp tile": the register / shared-memory image of one
// warp's chains, laid out so that a warp loads and stores it with coalesced 16-byte accesses:
//
//   bytes [   0,3072)  R image : 6 x float4 per lane, element [v][lane]; float f = 4v+e of a
//                                lane = coordinate (f%3) of the lane's bead f/3
//   bytes [3072,7168)  A image : [chain in warp][slot 0..N-1] float4 = (A_x, A_y, A_z, A_x low part);
//                                A_x + low part is the anchor's x, kept as a compensated sum so
//                                that the affine advection of eq (45) does not drift in fp32.
//                                Under a general tensor (ssm_step_kappa) the fourth word holds three
//                                signed 10-bit low parts instead, bits [10c, 10c + 10) for coordinate c
//                                in units of ulp(A_c) / 1024 (advect_packed in ssm_step.cu); the host
//                                tracks which encoding is current and clears the word on a change
//   bytes [7168,7424)  S image : [chain in warp][slot] uint8, 0 = empty, 1..N
//   bytes [7424,7552)  Z       : [chain in warp] int32 (32 entries, CPW used)
#pragma once
#include <cstdint>

// Device-side assertions of the checked build (python -m paper_1106_2899_b200.build --check -> libssm_check.so,
// loaded with SSM_LIB=check): every index the kernels form into the warp's shared memory and into the tiles is
// tested against its bounds, and a violation traps (the next CUDA call on the stream fails).  Compiled out of the
// product library.  (compute-sanitizer is closed on the B200 pool this was developed on; profiles/r2_sanitizers.md.)
#ifdef SSM_CHECK
#define SSM_ASSERT(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define SSM_ASSERT(cond) do { } while (0)
#endif

namespace ssm {

constexpr int kBPL = 8;                      // beads per lane
constexpr int kTileBytes = 7552;
constexpr int kTileR = 0, kTileA = 3072, kTileS = 7168, kTileZ = 7424;
constexpr int kWarpsPerBlock = 8;
constexpr int kBlockThreads = 32 * kWarpsPerBlock;
constexpr int kMaxFuse = 32;                 // time steps fused per launch (stress accumulators in smem)
constexpr int kFxShift = 26;                 // slip-spring displacement fixed point: 2^-26 b
constexpr int kStressShift = 18;             // ensemble stress fixed point: 2^-18 kT per lane share
constexpr int kSampleShift = 20;             // per-chain slip-spring virial (correlator samples): 2^-20

// per-warp shared memory of the step kernel.  The bead positions and the slip-spring force
// accumulators share one index: coordinate c of bead b of the warp (0..255) sits at word
//   3 b + 4 (b >> 5) + c      (a lane's 24 words are contiguous; 4 words of padding after every 4 lanes)
// so that the bead lanes move their 24 words as 6 aligned 16-byte accesses -- the lanes of a quarter warp start
// 96 bytes apart, the two halves of it a further 16: eight distinct 16-byte bank groups, conflict-free -- the
// position mirror is the lane's register image as it is, and, for chains of up to 32 beads (which never straddle
// a padding gap), the slot phase finds a bead's neighbours along the chain exactly 3 words away.  (An earlier
// layout padded every lane to 28 words: also conflict-free, but the neighbour offset then depended on the bead's
// place in its lane, a dozen issue slots per slot pass.)
constexpr int kSmRm = 0;         // float[800]  bead positions mirror (+1.3 kB spare up to kSmA)
constexpr int kSmA = 4608;       // float4[256] anchors [chain][slot] (x, y, z, x low part)
constexpr int kSmFx = 8704;      // int  [800]  fixed-point slip-spring displacement per bead coordinate (+0.4 kB spare up to kSmS)
constexpr int kSmS = 12288;      // uint8[256]  bead index per slot
constexpr int kSmZ = 12544;      // int  [32]   Z per chain
constexpr int kSmX = 12672;      // int  [33]   exclusive prefix of Z over the warp's chains (+ total), padded to 36
constexpr int kSmEv = 12816;     // uint [64]   construction candidates [chain][word]: bit k = attempt k passed the 16-bit test; [32 + chain] = (k << 16) | half of the chain's latest candidate
constexpr int kSmSamp = 13072;   // int  [32]   per-chain fixed-point sum of d_x d_y over slip-springs (sample steps)
constexpr int kSmKeys = 3840;    // uint [20]   the warp's copy of the Philox round keys (16-byte aligned)
constexpr int kSmKap = 3920;     // float[9]   dt kappa of the warp's group of chains (general flow only), up to 3956
constexpr int kSmPre = 3968;     // uint4[40]   what rounds 1, 2 of Philox make of (domain, chain) (ssm_rng.cuh, stream_prefix): [3][8] for the
                                 //             NOISE, SLOT and ATTEMPT domains of up to 8 chains per warp, [2][16] (NOISE, SLOT) of 16; up to 4608
constexpr int kSmSamp2 = 3584;   // int  [2][32] the same for d_y d_z and d_z d_x (isotropic correlator), in the spare kB after the mirror
constexpr int kStageSteps = 8;   // recorded steps whose warp sums wait in kSmStage before they are added to the CTA sums
constexpr int kSmStage = 13200;  // int  [8][12] warp sums of the last recorded steps (int32 fixed point)
constexpr int kSmDm = 13584;     // uint [32]   destruction masks [chain][word]: bit j = slip-spring j was destroyed in this step
constexpr int kSmMap = 13712;    // uint8[128]  dealing map: byte 4 lane + it = (chain << log2 N) | slot of the warp's
                                 //             slip-spring number lane + 32 it (it = 0..3), rebuilt when some Z changes
constexpr int kSmWarp = 13968;
constexpr int kSmAcc = kWarpsPerBlock * kSmWarp;                          // int64 [kMaxFuse][12] per CTA
constexpr int kSmStep = kSmAcc + kMaxFuse * 12 * 8;                       // 114,816 B: 2 CTAs per SM (2 x (114,816 + 1024) <= 233,472)
__host__ __device__ constexpr int fx_index(int bead_in_warp) { return bead_in_warp * 3 + ((bead_in_warp >> 5) << 2); }

struct StepParams {
    unsigned char *state;             // warp tiles
    long long     *stress;            // [capacity][12] int64 fixed-point sums; slot of this launch's first record
    float2        *samples;           // [n_sample_steps of this launch][n_comp][M] (f, g) per chain and component, or null
    int            n_comp;            // 1: xy; 3: xy, yz, zx
    long long      n_chains;          // M (chains >= M in the last tile are padding)
    unsigned long long chain_offset;  // global index of local chain 0
    unsigned long long step0;         // global index of the first step of this launch
    int            n_tiles;           // tiles this launch steps: [tile_first, tile_first + n_tiles)
    int            tile_first;
    int           *tile_counter;      // [2] in the workspace: tiles handed out beyond each warp's first; slot counter_slot is
    int            counter_slot;      // this launch's (zero on entry), the other one is zeroed for the next launch
    int            n_fuse;            // steps in this launch (<= kMaxFuse)
    unsigned       rec_mask;          // bit n: the ensemble stress is recorded after step n of this launch
    unsigned       smp_mask;          // bit n: the correlator is fed after step n of this launch
    int            n_rec;             // popcount(rec_mask)
    int            springs_on;
    int            k_attempts;        // 0: K = N - Z (GPU); k > 0: K = min(k, N - Z)
    int            n_act;             // N, the number of beads of a chain (<= 8G, the places a chain occupies)
    unsigned rk[20];  // Philox round keys: (k0 + r W0, k1 + r W1), r = 0..9
    float dt3;        // 3 dt                 (Rouse spring constant 3kT/b^2, eq 1)
    float bm_noise;   // -2 ln2 * 2 dt: r^2 = bm * log2(u) gives sqrt(2 dt) * N(0,1)  (eqs 44, 46, 47)
    float bm_anchor;  // -2 ln2 * N_s/3: anchor offsets of new slip-springs (eq 52)
    float gdt;        // shear_rate * dt      (eq 44, 45 with kappa_xy of eq 60)
    const float *kappa;               // null, or [groups][9] dt kappa_ab row-major (eqs 18, 21): general flow
    int   tiles_per_group;            // group of a warp tile = tile / tiles_per_group
    float fx_scale;   // dt * (3/N_s) * 2^kFxShift
    float q2l;        // 2 * (3/(4 N_s)) * log2(e): exponent scale of 1 - tanh(x) = 2/(1+e^{2x})
    float h2;         // 2 dt/zeta_s
    float cs;         // 3/N_s                (eq 76)
    unsigned t_destroy;               // T(min{dt/zeta_s, 1})                 (eq 53)
    unsigned t_c1[129], t_c2[129];    // T(p_c(K)), T(2 p_c(K)), K = 1..128   (eqs 50, 51)
    int h_c2[129];                    // the 23-bit code of attempt k is (h << 7) | e with a 16-bit h (reading R22):
                                      // h <= h_c2[K] = (T(2 p_c(K)) - 1) >> 7 is necessary for success (-1: never)
};

struct InitParams {
    unsigned char *state;
    long long      n_chains_padded;   // n_tiles * CPW
    long long      n_chains;          // M
    unsigned long long chain_offset;
    unsigned       rk[20];            // Philox round keys
    int            n_beads;           // N
    int            n_pad;             // 8G: bead places per chain in the tiles
    int            springs_on;
    float          bm_bond;           // -2 ln2 / 3:     bond components N(0, 1/3)    (eq 6)
    float          bm_anchor;         // -2 ln2 N_s / 3: anchor offsets N(0, N_s/3)  (eq 15)
    unsigned       t_cdf[128];        // T(P(Z <= z)), z = 0..zmax-1  (eq 12)
};

constexpr int kCorrMaxLevels = 32;
struct CorrParams {
    const float2 *samples;     // [n_samples][Mv] (f, g) = (sigma_ab, sigma_ab + sigma^(v)_ab); Mv = n_comp M histories,
                               // history q M + k = component q (xy, yz, zx) of chain k
    float *ring;               // [L][P][Mv] block-averaged g history
    float *acc_f, *acc_g;      // [L][Mv] first element of the pending pair
    long long *sum;            // [groups][L][P] int64 fixed point (2^-16): f_new g_old (eq 43)
    long long *sum_gg;         // [groups][L][P] int64 fixed point (2^-16): g_new g_old (eq 66)
    long long M;               // chains
    long long Mv;              // histories = n_comp * M
    unsigned long long chain_offset;
    int n_samples, L, Pb, groups;
    unsigned char pos[kCorrMaxLevels], filled[kCorrMaxLevels], parity[kCorrMaxLevels];   // at launch start
};

// What an entry point defined outside ssm_api.cu (ssm_noalloc.cu) may see of a ctx, whose struct is private to
// ssm_api.cu: the tiled state, the chain geometry, 3/N_s and the stream.  ctx_view fills it; ctx_fail records an
// error text on the ctx (or on the thread when ctx is null) and returns the code; ctx_add_launches keeps
// ssm_launch_count honest.
struct CtxView {
    const unsigned char *state;   // warp tiles (device)
    int       n_beads;            // N
    long long n_chains;           // M
    float     cs;                 // 3/N_s (eq 76)
    void     *stream;             // cudaStream_t
};

// address of bead coordinate / slot entry inside the tiled state (host and device)
__host__ __device__ inline int padded_beads(int n) { int g = kBPL; while (g < n) g <<= 1; return g; }
__host__ __device__ inline int chains_per_warp(int n_beads) { return 256 / n_beads; }
__host__ __device__ inline long long off_R(long long chain, int n_beads, int bead, int c)
{
    const int G = n_beads / kBPL, cpw = 32 / G;
    const long long tile = chain / cpw; const int cw = (int)(chain % cpw);
    const int lane = cw * G + bead / kBPL, f = (bead % kBPL) * 3 + c;
    return tile * kTileBytes + kTileR + (((f >> 2) * 32 + lane) * 4 + (f & 3)) * 4;
}
__host__ __device__ inline long long off_A(long long chain, int n_beads, int slot, int c /* 0..3 */)
{
    const int cpw = 256 / n_beads;
    return (chain / cpw) * kTileBytes + kTileA + (((int)(chain % cpw) * n_beads + slot) * 4 + c) * 4;
}
__host__ __device__ inline long long off_S(long long chain, int n_beads, int slot)
{
    const int cpw = 256 / n_beads;
    return (chain / cpw) * kTileBytes + kTileS + (int)(chain % cpw) * n_beads + slot;
}
__host__ __device__ inline long long off_Z(long long chain, int n_beads)
{
    const int cpw = 256 / n_beads;
    return (chain / cpw) * kTileBytes + kTileZ + (int)(chain % cpw) * 4;
}

}  // namespace ssm
