/*
 * ssm_oracle.h -- declarations of the fp64 CPU oracle (see ssm_oracle.c).
 * TEST INFRASTRUCTURE ONLY: used by tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs.  Not part of the product, not included by it.
 */
#ifndef SSM_ORACLE_H
#define SSM_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Philox stream domains */
enum {
    ORACLE_DOM_NOISE = 0,       /* step noise: normal m = 3*bead + axis = normal m&7 of call m>>3 */
    ORACLE_DOM_SLOT = 1,        /* call j>>1: words 2(j&1), 2(j&1)+1 = u_hop, u_end of j  */
    ORACLE_DOM_ATTEMPT = 2,     /* call k>>3: half k&1 of word (k&7)>>1 = high 16 bits of the 23-bit code of attempt k */
    ORACLE_DOM_ANCHOR = 3,      /* call k: normals 0..2 (words 0, 1) = anchor offset of attempt k; top 7 bits of word 2 =
                                   low 7 bits of its 23-bit code */
    ORACLE_DOM_INIT_BOND = 4,   /* step 0: normal m = 3*bond + axis                       */
    ORACLE_DOM_INIT_Z = 5,      /* step 0, call 0, word 0 -> Z                            */
    ORACLE_DOM_INIT_SLOT = 6,   /* step 0, call j, word 0 -> S_j                          */
    ORACLE_DOM_INIT_ANCHOR = 7  /* step 0, call j: normals 0..2 -> anchor offset          */
};
/* k_mode: K of eqs (50),(51), "an integer parameter which can depend on Z":
 * 0 = K = z_max - Z (the paper's GPU choice); k > 0 = K = min(k, z_max - Z)
 * (k = 1 is the paper's CPU choice). */
enum { ORACLE_K_EMPTY = 0, ORACLE_K_ONE = 1 };

typedef struct {
    int32_t  n_beads;      /* N */
    int64_t  n_chains;     /* M */
    int32_t  z_max;        /* 0 -> N */
    double   n_s, n_0, zeta_s, dt;
    uint64_t seed;
    int32_t  k_mode;
    uint64_t chain_offset; /* global index of local chain 0 (Philox is keyed by the global index) */
    int32_t  noise_bits;   /* resolution of the Box-Muller inputs behind the bead noise w_i (eqs 46, 47; DESIGN.md
                              reading R24).  0 or 16: the RNG contract shared with the GPU (16-bit codes, one word per
                              pair of normals, eight normals per call).  23: the full-resolution law this oracle was
                              first written with (23-bit uniforms, two words per pair, four normals per call: normal
                              m = 3*bead + axis is normal m&3 of call m>>2).  23 has no GPU counterpart; it exists so
                              that the tests can show that the dynamics do not depend on the narrowing (the A/B pin
                              of tests/test_oracle_noise_law.py) */
} oracle_params;

typedef struct {
    double  *R;                  /* [M][N][3]     */
    double  *A;                  /* [M][zmax][3]  */
    int32_t *S;                  /* [M][zmax], 1..N, first Z entries occupied, rest 0 */
    int32_t *Z;                  /* [M]           */
    int64_t  step;               /* global step counter */
    int64_t *first_fragile_step; /* [M], -1 = none */
    double  *min_margin;         /* [M] */
} oracle_state;

typedef struct {
    int64_t n_chains; int levels, bins, groups;
    int n_comp;                    /* 1: xy only; 3: xy, yz, zx feed the same sums (isotropic average) */
    double *ring; int *pos, *filled; double *acc_f, *acc_g; int *acc_n;
    double *sum; int64_t *count;   /* [groups][levels][bins]: sum of f_new g_old (eq 43) */
    double *sum_gg;                /* [groups][levels][bins]: sum of g_new g_old (eq 66) */
} oracle_corr;

void     oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void     oracle_stream(uint64_t seed, int domain, uint64_t step, uint64_t chain, uint32_t item, uint32_t out[4]);
uint32_t oracle_code23(uint32_t w);
double   oracle_u23(uint32_t w);
int64_t  oracle_threshold23(double p);
void     oracle_box_muller(uint32_t w, double z[2]);
void     oracle_box_muller23(uint32_t wa, uint32_t wb, double z[2]);
double   oracle_stream_normal(uint64_t seed, int domain, uint64_t step, uint64_t chain, uint32_t m);
int      oracle_zmax(const oracle_params *p);
void     oracle_hop_probabilities(const oracle_params *p, const double *R, const double *A, int s,
                                  double *p_plus, double *p_minus);
void     oracle_chain_stress(const oracle_params *p, const double *R, const double *A, const int32_t *S,
                             int Z, double sig[6], double sigv[6]);
void     oracle_poisson_thresholds(const oracle_params *p, int64_t *tcdf);
void     oracle_init_chain(const oracle_params *p, uint64_t chain, double *R, double *A, int32_t *S, int32_t *Z);
void     oracle_step_chain(const oracle_params *p, uint64_t chain, uint64_t step, double shear_rate,
                           double *R, double *A, int32_t *S, int32_t *Z, double *min_margin);
void     oracle_step_chain_kappa(const oracle_params *p, uint64_t chain, uint64_t step, const double kappa[9],
                                 double *R, double *A, int32_t *S, int32_t *Z, double *min_margin);
oracle_corr *oracle_corr_create(int64_t n_chains, int levels, int bins, int groups);
oracle_corr *oracle_corr_create_iso(int64_t n_chains, int levels, int bins, int groups, int n_comp);
void     oracle_corr_destroy(oracle_corr *c);
void     oracle_corr_push(oracle_corr *c, int64_t chain_local, int group, double f, double g);
void     oracle_corr_sums(const oracle_corr *c, double *sum, double *sum_gg, int64_t *count);
int      oracle_corr_result(const oracle_corr *c, int n_beads, double base_dt, int cap,
                            double *lag_time, double *G, double *se);
int      oracle_corr_result_virtual(const oracle_corr *c, double base_dt, int cap,
                                    double *lag_time, double *dGv, double *se);
int64_t  oracle_run(const oracle_params *p, oracle_state *st, int64_t n_steps, double shear_rate,
                    int stress_every, double *stress_out, int sample_every, oracle_corr *corr,
                    double guard, int n_threads);
int64_t  oracle_run_kappa(const oracle_params *p, oracle_state *st, int64_t n_steps, int64_t chains_per_group,
                          const double *kappa, int stress_every, double *stress_out, int sample_every,
                          oracle_corr *corr, double guard, int n_threads);

#ifdef __cplusplus
}
#endif
#endif
