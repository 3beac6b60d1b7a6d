/*
 * ssm_oracle.c -- fp64 CPU ORACLE for the single-chain slip-spring model of
 * T. Uneyama (arxiv 1106.2899).  P:Lnnn = /root/reference/PAPER.md line nnn.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or constant generator with the CUDA path under paper_1106_2899_b200/.
 *
 * It is the algorithm of P:L286-L362 (section 3.1) written out step by step in the
 * paper's order and notation, in double precision, one chain at a time:
 *
 *   substep 1  explicit Euler for R_i and A_j            eqs (44),(45)
 *   substep 2  Glauber hop of every S_j                  eqs (22)-(24)  P:L161-L172,
 *                                                        eqs (48),(49)
 *   substep 3  construction / destruction at chain ends  eqs (50)-(53)
 *   observables  sigma eq (16), sigma^(v) eq (76), mean eq (54)
 *   G(t)        eq (43) P:L277 through a per-chain multi-tau correlator
 *   initial state  equilibrium sampling eq (13)
 *
 * Units b = kT = zeta = 1.  Readings of garbled/silent passages are listed in
 * DESIGN.md section 3 ("R1".."R20"); each is cited where it is used below.
 *
 * Random numbers: the paper's LCG is replaced by the counter-based
 * Philox4x32-10 (Salmon et al., SC'11) as BASELINE.json's north_star directs; the
 * stream layout is the "RNG contract" of DESIGN.md section 4 and is restated here.
 *
 * Parity unpinned: the exact finite-dt stationary law WITH slip-springs (only O(dt)
 * close to eqs 12-15) and the curves of Figs 1-8 (images absent).  Everything else is
 * pinned by tests/test_oracle_*.py.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <pthread.h>

#include "ssm_oracle.h"

/* ------------------------------------------------------------------------- */
/* Philox4x32-10: 10 rounds; round: (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2),    */
/* hi(M0*c0)^c3^k1, lo(M0*c0)); key += (W0,W1) between rounds.                        */
/* ------------------------------------------------------------------------- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* RNG contract: key = (seed lo, seed hi);
 * counter = (step lo 32, domain<<28 | step bits 32..59, global chain index, item). */
void oracle_stream(uint64_t seed, int domain, uint64_t step, uint64_t chain, uint32_t item,
                   uint32_t out[4])
{
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { (uint32_t)step,
                        ((uint32_t)domain << 28) | (uint32_t)((step >> 32) & 0x0FFFFFFFu),
                        (uint32_t)chain, item };
    oracle_philox4x32_10(ctr, key, out);
}

/* 23-bit code of a word and the uniform it stands for: u = (k + 1/2) 2^-23 in (0,1). */
uint32_t oracle_code23(uint32_t w) { return w >> 9; }
double   oracle_u23(uint32_t w)    { return ((double)(w >> 9) + 0.5) * 0x1p-23; }

/* "u < p"  <=>  k < T(p),  T(p) = ceil(p 2^23 - 1/2)   (u = (k+1/2) 2^-23, k integer) */
int64_t oracle_threshold23(double p)
{
    double t = ceil(p * 8388608.0 - 0.5);
    if (t < 0.0) t = 0.0;
    if (t > 8388608.0) t = 8388608.0;
    return (int64_t)t;
}

/* Box-Muller on one Philox word (reading R24): the low and the high
 * half of the word are two 16-bit codes ka, kb; u_a = (ka + 1/2) 2^-16, u_b = (kb + 1/2) 2^-16;
 * r = sqrt(-2 ln u_a), theta = 2 pi (u_b - 1/2); (z0, z1) = (r cos theta, r sin theta).
 * |z| <= sqrt(34 ln 2) = 4.86; E[z^2] = 1 - 5e-6 (pinned by enumeration in the tests). */
void oracle_box_muller(uint32_t w, double z[2])
{
    double ua = ((double)(w & 0xFFFFu) + 0.5) * 0x1p-16;
    double ub = ((double)(w >> 16) + 0.5) * 0x1p-16;
    double r = sqrt(-2.0 * log(ua));
    double th = 6.283185307179586476925286766559 * (ub - 0.5);
    z[0] = r * cos(th);
    z[1] = r * sin(th);
}

/* The same transform at the full resolution of the decision uniforms (P:L307 fixes no resolution): two
 * words give one pair, u_a, u_b = (k + 1/2) 2^-23; |z| <= sqrt(48 ln 2) = 5.77.  Used only when
 * oracle_params.noise_bits = 23 (the A/B pin of reading R24); the contract with the GPU is the 16-bit form. */
void oracle_box_muller23(uint32_t wa, uint32_t wb, double z[2])
{
    double ua = oracle_u23(wa), ub = oracle_u23(wb);
    double r = sqrt(-2.0 * log(ua));
    double th = 6.283185307179586476925286766559 * (ub - 0.5);
    z[0] = r * cos(th);
    z[1] = r * sin(th);
}

/* Normal number m of the stream (domain, step, chain): Philox call q = m>>3 gives the
 * eight normals z_{8q+2e}, z_{8q+2e+1} from word e = 0..3. */
static void normal_call(uint64_t seed, int domain, uint64_t step, uint64_t chain, uint32_t q,
                        double z[8])
{
    uint32_t w[4];
    oracle_stream(seed, domain, step, chain, q, w);
    for (int e = 0; e < 4; ++e) oracle_box_muller(w[e], z + 2 * e);
}
double oracle_stream_normal(uint64_t seed, int domain, uint64_t step, uint64_t chain, uint32_t m)
{
    double z[8];
    normal_call(seed, domain, step, chain, m >> 3, z);
    return z[m & 7];
}

/* ------------------------------------------------------------------------- */
/* parameters                                                                  */
/* ------------------------------------------------------------------------- */
static int springs_on(const oracle_params *p) { return p->n_0 > 0.0 && isfinite(p->n_0); }
int oracle_zmax(const oracle_params *p) { return p->z_max > 0 ? p->z_max : p->n_beads; }

/* Glauber hop probabilities, eqs (23),(24) with the cap of eqs (48),(49) (reading R5):
 * p+- = min{ (dt/zeta_s) [1 - tanh( (3/4N_s) (|R_{s+-1}-A|^2 - |R_s-A|^2) )], 1/2 },
 * 0 beyond the chain ends.  R is the chain's [N][3], s is 1-based. */
void oracle_hop_probabilities(const oracle_params *p, const double *R, const double *A, int s,
                              double *p_plus, double *p_minus)
{
    const int N = p->n_beads;
    const double h = p->dt / p->zeta_s, q = 3.0 / (4.0 * p->n_s);
    double e0 = 0, ep = 0, em = 0;
    for (int c = 0; c < 3; ++c) {
        double d = R[3 * (s - 1) + c] - A[c];
        e0 += d * d;
    }
    *p_plus = 0.0; *p_minus = 0.0;
    if (s < N) {
        for (int c = 0; c < 3; ++c) { double d = R[3 * s + c] - A[c]; ep += d * d; }
        *p_plus = fmin(h * (1.0 - tanh(q * (ep - e0))), 0.5);
    }
    if (s > 1) {
        for (int c = 0; c < 3; ++c) { double d = R[3 * (s - 2) + c] - A[c]; em += d * d; }
        *p_minus = fmin(h * (1.0 - tanh(q * (em - e0))), 0.5);
    }
}

/* sigma (eq 16) and sigma^(v) (eq 76; reading R11,R12) of one chain.
 * component order xx,yy,zz,xy,yz,zx. */
void oracle_chain_stress(const oracle_params *p, const double *R, const double *A, const int32_t *S,
                         int Z, double sig[6], double sigv[6])
{
    const int N = p->n_beads;
    static const int ca[6] = {0, 1, 2, 0, 1, 2}, cb[6] = {0, 1, 2, 1, 2, 0};
    for (int t = 0; t < 6; ++t) { sig[t] = 0.0; sigv[t] = 0.0; }
    for (int i = 0; i + 1 < N; ++i)
        for (int t = 0; t < 6; ++t)
            sig[t] += 3.0 * (R[3 * (i + 1) + ca[t]] - R[3 * i + ca[t]])
                          * (R[3 * (i + 1) + cb[t]] - R[3 * i + cb[t]]);
    for (int t = 0; t < 3; ++t) sig[t] -= (double)N;
    for (int j = 0; j < Z; ++j) {
        const double *r = R + 3 * (S[j] - 1), *a = A + 3 * j;
        for (int t = 0; t < 6; ++t)
            sigv[t] += (3.0 / p->n_s) * (r[ca[t]] - a[ca[t]]) * (r[cb[t]] - a[cb[t]]);
    }
    for (int t = 0; t < 3; ++t) sigv[t] -= (double)Z;
}

/* ------------------------------------------------------------------------- */
/* equilibrium initial state, eq (13): one chain                 */
/* ------------------------------------------------------------------------- */
/* Poisson(N/N0) CDF thresholds (eq 12): Tcdf[z] = T(P(Z<=z)), z = 0..zmax-1 */
void oracle_poisson_thresholds(const oracle_params *p, int64_t *tcdf)
{
    const int zmax = oracle_zmax(p);
    const double lam = (double)p->n_beads / p->n_0;
    double pmf = exp(-lam), cdf = 0.0;
    for (int z = 0; z < zmax; ++z) {
        if (z > 0) pmf = pmf * lam / (double)z;
        cdf += pmf;
        tcdf[z] = oracle_threshold23(cdf);
    }
}

void oracle_init_chain(const oracle_params *p, uint64_t chain, double *R, double *A, int32_t *S, int32_t *Zout)
{
    const int N = p->n_beads, zmax = oracle_zmax(p);
    /* 1. Gaussian bonds, variance b^2/3 per axis (eq 6); R_1 = 0 (reading R15) */
    R[0] = R[1] = R[2] = 0.0;
    double z8[8];
    for (int i = 0; i + 1 < N; ++i)
        for (int c = 0; c < 3; ++c) {
            uint32_t m = (uint32_t)(3 * i + c);
            if ((m & 7) == 0) normal_call(p->seed, ORACLE_DOM_INIT_BOND, 0, chain, m >> 3, z8);
            R[3 * (i + 1) + c] = R[3 * i + c] + sqrt(1.0 / 3.0) * z8[m & 7];
        }
    /* 2. Z ~ Poisson(N/N0) clamped at zmax (eq 12; reading R7) by inversion in the
     *    integer domain */
    int Z = 0;
    if (springs_on(p)) {
        int64_t *tcdf = (int64_t *)malloc(sizeof(int64_t) * (size_t)zmax);
        oracle_poisson_thresholds(p, tcdf);
        uint32_t w[4];
        oracle_stream(p->seed, ORACLE_DOM_INIT_Z, 0, chain, 0, w);
        int64_t k = (int64_t)oracle_code23(w[0]);
        while (Z < zmax && k >= tcdf[Z]) ++Z;
        free(tcdf);
    }
    /* 3. S_j uniform on 1..N (eq 14), A_j Gaussian about R_{S_j}, variance N_s/3 per
     *    axis (eq 15) */
    for (int j = 0; j < zmax; ++j) { S[j] = 0; A[3 * j] = A[3 * j + 1] = A[3 * j + 2] = 0.0; }
    for (int j = 0; j < Z; ++j) {
        uint32_t w[4];
        oracle_stream(p->seed, ORACLE_DOM_INIT_SLOT, 0, chain, (uint32_t)j, w);
        S[j] = 1 + (int)(((uint64_t)w[0] * (uint64_t)N) >> 32);
        normal_call(p->seed, ORACLE_DOM_INIT_ANCHOR, 0, chain, (uint32_t)j, z8);
        for (int c = 0; c < 3; ++c)
            A[3 * j + c] = R[3 * (S[j] - 1) + c] + sqrt(p->n_s / 3.0) * z8[c];
    }
    *Zout = Z;
}

/* ------------------------------------------------------------------------- */
/* one time step of one chain                                     */
/* ------------------------------------------------------------------------- */
/* K of eqs (50),(51): number of construction attempts (reading R9) */
static int attempts_K(const oracle_params *p, int Z)
{
    const int empty = oracle_zmax(p) - Z;
    if (!springs_on(p) || empty <= 0) return 0;
    if (p->k_mode > 0) return p->k_mode < empty ? p->k_mode : empty;   /* fixed K (K = 1: the paper's CPU choice) */
    return empty;                                                      /* K = N - Z: the paper's GPU choice */
}

/* One time step of one chain.  kappa == NULL: simple shear kappa_xy = shear_rate (eq 60);
 * else kappa[3a + b] = kappa_ab is the full velocity gradient tensor of eqs (18), (21)
 * and shear_rate is ignored. */
static void step_chain(const oracle_params *p, uint64_t chain, uint64_t step, double shear_rate, const double *kappa,
                       double *R, double *A, int32_t *S, int32_t *Zio, double *min_margin)
{
    const int N = p->n_beads;
    const double dt = p->dt, h = dt / p->zeta_s;
    int Z = *Zio;
    double *F = (double *)malloc(sizeof(double) * 3 * (size_t)N);

    /* ---- substep 1: forces -dJ/dR_i from time-t values (eq 1, eq 18; readings R2,R3) */
    for (int i = 0; i < N; ++i)
        for (int c = 0; c < 3; ++c) {
            double f = 0.0;
            if (i + 1 < N) f += 3.0 * (R[3 * (i + 1) + c] - R[3 * i + c]);
            if (i > 0)     f -= 3.0 * (R[3 * i + c] - R[3 * (i - 1) + c]);
            F[3 * i + c] = f;
        }
    for (int j = 0; j < Z; ++j) {
        int s = S[j] - 1;
        for (int c = 0; c < 3; ++c) F[3 * s + c] -= (3.0 / p->n_s) * (R[3 * s + c] - A[3 * j + c]);
    }
    /* explicit Euler, eqs (44),(45) (reading R1); the affine term dt kappa . R_i, dt kappa . A_j uses the
     * time-t positions; kappa_xy = shear_rate only (eq 60) when no tensor is given */
    double z8[8];
    for (int i = 0; i < N; ++i) {
        const double rx = R[3 * i], ry = R[3 * i + 1], rz = R[3 * i + 2];
        for (int c = 0; c < 3; ++c) {
            uint32_t m = (uint32_t)(3 * i + c);
            double w;                                   /* w_i of eqs (46), (47) */
            if (p->noise_bits == 23) {                  /* full-resolution law (A/B pin of reading R24 only) */
                if ((m & 3) == 0) {
                    uint32_t wd[4];
                    oracle_stream(p->seed, ORACLE_DOM_NOISE, step, chain, m >> 2, wd);
                    oracle_box_muller23(wd[0], wd[1], z8);
                    oracle_box_muller23(wd[2], wd[3], z8 + 2);
                }
                w = z8[m & 3];
            } else {
                if ((m & 7) == 0) normal_call(p->seed, ORACLE_DOM_NOISE, step, chain, m >> 3, z8);
                w = z8[m & 7];
            }
            double flow;
            if (kappa) flow = dt * (kappa[3 * c] * rx + kappa[3 * c + 1] * ry + kappa[3 * c + 2] * rz);
            else flow = (c == 0) ? dt * shear_rate * ry : 0.0;
            R[3 * i + c] = R[3 * i + c] + dt * F[3 * i + c] + flow + sqrt(2.0 * dt) * w;
        }
    }
    for (int j = 0; j < Z; ++j) {
        if (kappa) {
            const double ax = A[3 * j], ay = A[3 * j + 1], az = A[3 * j + 2];
            for (int c = 0; c < 3; ++c)
                A[3 * j + c] = A[3 * j + c] + dt * (kappa[3 * c] * ax + kappa[3 * c + 1] * ay + kappa[3 * c + 2] * az);
        } else A[3 * j] = A[3 * j] + dt * shear_rate * A[3 * j + 1];
    }
    free(F);

    /* ---- substep 2: hop, one uniform per slip-spring, cumulative intervals
     *      [0,p+) -> S+1, [p+,p+ + p-) -> S-1 (readings R4,R5,R6); strict "<" */
    for (int j = 0; j < Z; ++j) {
        uint32_t w[4];
        oracle_stream(p->seed, ORACLE_DOM_SLOT, step, chain, (uint32_t)(j >> 1), w);
        double u = oracle_u23(w[2 * (j & 1)]);
        double pp, pm;
        oracle_hop_probabilities(p, R, A + 3 * j, S[j], &pp, &pm);
        if (min_margin) {
            double m1 = fabs(u - pp), m2 = fabs(u - (pp + pm));
            double m = m1 < m2 ? m1 : m2;
            if (m < *min_margin) *min_margin = m;
        }
        if (u < pp) S[j] += 1;
        else if (u < pp + pm) S[j] -= 1;
    }

    /* ---- substep 3: reconstruction at the chain ends (readings R7,R8,R9).
     * A slip-spring is exposed to destruction only if it existed before this substep;
     * K is taken from the Z before this substep. */
    const int Z0 = Z;
    const int K = attempts_K(p, Z0);
    /* destruction, eq (53): prob min{(dt/zeta_s)(delta_{S,1}+delta_{S,N}), 1}.
     * "We reset indices of slip-springs after the constructions or destructions" so that
     * they run from 1 to Z; the paper does not say in which order, and
     * slip-springs are indistinguishable (eq 2), so (reading R21) the
     * slip-springs are visited from the last to the first and a destroyed one is replaced
     * by the one that is last at that moment (already visited, hence a survivor). */
    const int64_t Td = oracle_threshold23(fmin(h, 1.0));
    int Zs = Z0;
    for (int j = Z0 - 1; j >= 0; --j) {
        int destroyed = 0;
        if (S[j] == 1 || S[j] == N) {
            uint32_t w[4];
            oracle_stream(p->seed, ORACLE_DOM_SLOT, step, chain, (uint32_t)(j >> 1), w);
            destroyed = (int64_t)oracle_code23(w[2 * (j & 1) + 1]) < Td;
        }
        if (destroyed) {
            --Zs;
            S[j] = S[Zs];
            for (int c = 0; c < 3; ++c) A[3 * j + c] = A[3 * Zs + c];
        }
    }
    /* construction, eqs (50)-(52): K attempts, each end with prob min{h/(N0 K), 1/2} */
    if (K > 0) {
        const double pc = fmin(h / (p->n_0 * (double)K), 0.5);
        const int64_t T1 = oracle_threshold23(pc), T2 = oracle_threshold23(2.0 * pc);
        uint32_t w[4] = {0, 0, 0, 0};
        for (int k = 0; k < K; ++k) {
            /* uniform of attempt k (reading R22): u = (code + 1/2) 2^-23 with the 23-bit
             * code = (h << 7) | e; h = 16-bit half (k&1) of word (k&7)>>1 of ATTEMPT call k>>3,
             * e = top 7 bits of word 2 of ANCHOR call k (whose words 0, 1 give the anchor offset) */
            uint32_t wa[4];
            if ((k & 7) == 0) oracle_stream(p->seed, ORACLE_DOM_ATTEMPT, step, chain, (uint32_t)(k >> 3), w);
            oracle_stream(p->seed, ORACLE_DOM_ANCHOR, step, chain, (uint32_t)k, wa);
            uint32_t h = (w[(k & 7) >> 1] >> (16 * (k & 1))) & 0xFFFFu;
            int64_t code = (int64_t)((h << 7) | (wa[2] >> 25));
            int snew = 0;
            if (code < T1) snew = 1;
            else if (code < T2) snew = N;
            if (snew) {
                normal_call(p->seed, ORACLE_DOM_ANCHOR, step, chain, (uint32_t)k, z8);
                S[Zs] = snew;
                for (int c = 0; c < 3; ++c)
                    A[3 * Zs + c] = R[3 * (snew - 1) + c] + sqrt(p->n_s / 3.0) * z8[c];
                ++Zs;
            }
        }
    }
    for (int j = Zs; j < oracle_zmax(p); ++j) { S[j] = 0; A[3 * j] = A[3 * j + 1] = A[3 * j + 2] = 0.0; }
    *Zio = Zs;
}

void oracle_step_chain(const oracle_params *p, uint64_t chain, uint64_t step, double shear_rate,
                       double *R, double *A, int32_t *S, int32_t *Zio, double *min_margin)
{
    step_chain(p, chain, step, shear_rate, NULL, R, A, S, Zio, min_margin);
}

/* the same step under a general velocity gradient tensor kappa[3a + b] = kappa_ab (eqs 18, 21) */
void oracle_step_chain_kappa(const oracle_params *p, uint64_t chain, uint64_t step, const double kappa[9],
                             double *R, double *A, int32_t *S, int32_t *Zio, double *min_margin)
{
    step_chain(p, chain, step, 0.0, kappa, R, A, S, Zio, min_margin);
}

/* ------------------------------------------------------------------------- */
/* multi-tau correlator (BASELINE.json config 2)          */
/* per chain: levels x bins ring of g = sigma_xy + sigma^(v)_xy; products       */
/* f_new * g_old with f = sigma_xy (eq 43, reading R14)                         */
/* ------------------------------------------------------------------------- */
static void corr_insert(oracle_corr *c, int64_t chain_local, int group, int lev, double f, double g)
{
    const int L = c->levels, P = c->bins, m = 2;
    if (lev >= L) return;
    double *ring = c->ring + ((size_t)chain_local * L + lev) * P;
    int *pos = c->pos + (size_t)chain_local * L + lev;
    int *fil = c->filled + (size_t)chain_local * L + lev;
    ring[*pos] = g;
    if (*fil < P) ++*fil;
    const int kmin = lev == 0 ? 0 : P / m;
    double *C = c->sum + ((size_t)group * L + lev) * P;
    double *C2 = c->sum_gg + ((size_t)group * L + lev) * P;
    int64_t *cnt = c->count + ((size_t)group * L + lev) * P;
    for (int k = kmin; k < P && k < *fil; ++k) {
        int idx = *pos - k; if (idx < 0) idx += P;
        C[k] += f * ring[idx];
        C2[k] += g * ring[idx];           /* for the virtual-stress contribution, eq (66) */
        cnt[k] += 1;
    }
    *pos = (*pos + 1) % P;
    double *af = c->acc_f + (size_t)chain_local * L + lev;
    double *ag = c->acc_g + (size_t)chain_local * L + lev;
    int *an = c->acc_n + (size_t)chain_local * L + lev;
    *af += f; *ag += g; ++*an;
    if (*an == m) {
        double mf = *af / m, mg = *ag / m;
        *af = 0.0; *ag = 0.0; *an = 0;
        corr_insert(c, chain_local, group, lev + 1, mf, mg);
    }
}

/* n_comp = 1: the xy component only (eq 43 as printed).  n_comp = 3: xy, yz and zx each keep their own
 * history and all feed the same sums -- the equilibrium ensemble is isotropic (eq 13 has no preferred
 * axis), so G_xyxy = G_yzyz = G_zxzx and the average is an estimate of the same G from three times
 * the data.  History slot of (chain k, component q) = q n_chains + k. */
oracle_corr *oracle_corr_create_iso(int64_t n_chains, int levels, int bins, int groups, int n_comp)
{
    oracle_corr *c = (oracle_corr *)calloc(1, sizeof(oracle_corr));
    c->n_chains = n_chains; c->levels = levels; c->bins = bins; c->groups = groups; c->n_comp = n_comp;
    size_t nl = (size_t)n_chains * n_comp * levels;
    c->ring = (double *)calloc(nl * bins, sizeof(double));
    c->pos = (int *)calloc(nl, sizeof(int));
    c->filled = (int *)calloc(nl, sizeof(int));
    c->acc_f = (double *)calloc(nl, sizeof(double));
    c->acc_g = (double *)calloc(nl, sizeof(double));
    c->acc_n = (int *)calloc(nl, sizeof(int));
    c->sum = (double *)calloc((size_t)groups * levels * bins, sizeof(double));
    c->sum_gg = (double *)calloc((size_t)groups * levels * bins, sizeof(double));
    c->count = (int64_t *)calloc((size_t)groups * levels * bins, sizeof(int64_t));
    return c;
}
oracle_corr *oracle_corr_create(int64_t n_chains, int levels, int bins, int groups)
{
    return oracle_corr_create_iso(n_chains, levels, bins, groups, 1);
}
void oracle_corr_destroy(oracle_corr *c)
{
    if (!c) return;
    free(c->ring); free(c->pos); free(c->filled); free(c->acc_f); free(c->acc_g); free(c->acc_n);
    free(c->sum); free(c->sum_gg); free(c->count); free(c);
}
void oracle_corr_push(oracle_corr *c, int64_t chain_local, int group, double f, double g)
{
    corr_insert(c, chain_local, group, 0, f, g);
}
/* raw accumulators [groups][levels][bins] (sum of f_new g_old, of g_new g_old, product counts), so that a test can
 * compare another correlator's sums bin by bin */
void oracle_corr_sums(const oracle_corr *c, double *sum, double *sum_gg, int64_t *count)
{
    const size_t n = (size_t)c->groups * c->levels * c->bins;
    memcpy(sum, c->sum, n * sizeof(double));
    memcpy(sum_gg, c->sum_gg, n * sizeof(double));
    memcpy(count, c->count, n * sizeof(int64_t));
}

/* distinct lags in increasing order: level 0 bins 0..P-1, level l>0 bins P/2..P-1.
 * G/(rho0 kT) = sum/(count N) (reading R13); se = std over groups / sqrt(groups). */
int oracle_corr_result(const oracle_corr *c, int n_beads, double base_dt, int cap,
                       double *lag_time, double *G, double *se)
{
    const int L = c->levels, P = c->bins, Gn = c->groups;
    int n = 0;
    for (int lev = 0; lev < L; ++lev)
        for (int k = (lev == 0 ? 0 : P / 2); k < P; ++k) {
            double s = 0.0; int64_t cn = 0;
            for (int g = 0; g < Gn; ++g) {
                s += c->sum[((size_t)g * L + lev) * P + k];
                cn += c->count[((size_t)g * L + lev) * P + k];
            }
            if (cn == 0) continue;
            if (n >= cap) return -1;
            lag_time[n] = (double)k * ldexp(1.0, lev) * base_dt;
            G[n] = s / ((double)cn * n_beads);
            if (se) {
                double mean = 0.0, var = 0.0; int used = 0;
                for (int g = 0; g < Gn; ++g) {
                    int64_t cg = c->count[((size_t)g * L + lev) * P + k];
                    if (cg > 0) { mean += c->sum[((size_t)g * L + lev) * P + k] / ((double)cg * n_beads); ++used; }
                }
                if (used > 1) {
                    mean /= used;
                    for (int g = 0; g < Gn; ++g) {
                        int64_t cg = c->count[((size_t)g * L + lev) * P + k];
                        if (cg > 0) {
                            double v = c->sum[((size_t)g * L + lev) * P + k] / ((double)cg * n_beads) - mean;
                            var += v * v;
                        }
                    }
                    se[n] = sqrt(var / (used - 1) / used);
                } else se[n] = NAN;
            }
            ++n;
        }
    return n;
}

/* Relative contribution of the virtual stress to the relaxation modulus, eq (66) P:L438:
 *   dGv(t) = [<sv(t) s(0)> + <sv(t) sv(0)>] / [<s(t) s(0)> + <s(t) sv(0)>],  s = sigma_xy, sv = sigma^(v)_xy.
 * With g = s + sv the denominator is <s(t) g(0)> (the sums of eq 43) and the numerator is
 * <sv(t) g(0)> = <g(t) g(0)> - <s(t) g(0)>.  se = std over groups of the per-group ratio / sqrt(groups). */
int oracle_corr_result_virtual(const oracle_corr *c, double base_dt, int cap,
                               double *lag_time, double *dGv, double *se)
{
    const int L = c->levels, P = c->bins, Gn = c->groups;
    int n = 0;
    for (int lev = 0; lev < L; ++lev)
        for (int k = (lev == 0 ? 0 : P / 2); k < P; ++k) {
            double sfg = 0.0, sgg = 0.0; int64_t cn = 0;
            for (int g = 0; g < Gn; ++g) {
                size_t i = ((size_t)g * L + lev) * P + k;
                sfg += c->sum[i]; sgg += c->sum_gg[i]; cn += c->count[i];
            }
            if (cn == 0) continue;
            if (n >= cap) return -1;
            lag_time[n] = (double)k * ldexp(1.0, lev) * base_dt;
            dGv[n] = (sgg - sfg) / sfg;
            if (se) {
                double mean = 0.0, var = 0.0; int used = 0;
                for (int g = 0; g < Gn; ++g) {
                    size_t i = ((size_t)g * L + lev) * P + k;
                    if (c->count[i] > 0) { mean += (c->sum_gg[i] - c->sum[i]) / c->sum[i]; ++used; }
                }
                if (used > 1) {
                    mean /= used;
                    for (int g = 0; g < Gn; ++g) {
                        size_t i = ((size_t)g * L + lev) * P + k;
                        if (c->count[i] > 0) { double v = (c->sum_gg[i] - c->sum[i]) / c->sum[i] - mean; var += v * v; }
                    }
                    se[n] = sqrt(var / (used - 1) / used);
                } else se[n] = NAN;
            }
            ++n;
        }
    return n;
}

/* ------------------------------------------------------------------------- */
/* ensemble driver: advance chains [k0,k1) by n_steps                          */
/* ------------------------------------------------------------------------- */
typedef struct {
    const oracle_params *p; oracle_state *st; int64_t k0, k1; int64_t n_steps; double shear_rate;
    int stress_every; double *stress_sum; /* [n_samples][12] partial */
    int sample_every; oracle_corr *corr; double guard;
    const double *kappa; int64_t chains_per_group;   /* kappa of local chain k: kappa + 9 (k / chains_per_group), or NULL */
} work_t;

static void *worker(void *arg)
{
    work_t *w = (work_t *)arg;
    const oracle_params *p = w->p; oracle_state *st = w->st;
    const int N = p->n_beads, zmax = oracle_zmax(p);
    for (int64_t k = w->k0; k < w->k1; ++k) {
        double *R = st->R + (size_t)k * N * 3, *A = st->A + (size_t)k * zmax * 3;
        int *S = st->S + (size_t)k * zmax;
        const uint64_t chain = p->chain_offset + (uint64_t)k;
        for (int64_t n = 0; n < w->n_steps; ++n) {
            const uint64_t step = (uint64_t)(st->step + n);
            double margin = INFINITY;
            step_chain(p, chain, step, w->shear_rate, w->kappa ? w->kappa + 9 * (k / w->chains_per_group) : NULL,
                       R, A, S, &st->Z[k], &margin);
            if (margin < st->min_margin[k]) st->min_margin[k] = margin;
            if (margin < w->guard && st->first_fragile_step[k] < 0) st->first_fragile_step[k] = (int64_t)step;
            const int64_t done = st->step + n + 1;          /* sample after the n-th step: t = n dt (R17) */
            const int rec = w->stress_every > 0 && done % w->stress_every == 0;
            const int smp = w->corr && w->sample_every > 0 && done % w->sample_every == 0;
            if (rec || smp) {
                double sig[6], sigv[6];
                oracle_chain_stress(p, R, A, S, st->Z[k], sig, sigv);
                if (rec) {
                    int64_t idx = done / w->stress_every - st->step / w->stress_every - 1;
                    double *o = w->stress_sum + (size_t)idx * 12;
                    for (int t = 0; t < 6; ++t) { o[t] += sig[t]; o[6 + t] += sigv[t]; }
                }
                if (smp)                                         /* components 3, 4, 5 = xy, yz, zx */
                    for (int q = 0; q < w->corr->n_comp; ++q)
                        oracle_corr_push(w->corr, (int64_t)q * w->corr->n_chains + k,
                                         (int)((chain / 32) % (uint64_t)w->corr->groups),
                                         sig[3 + q], sig[3 + q] + sigv[3 + q]);
            }
        }
    }
    return NULL;
}

/* stress_out: [n_samples][12] ensemble MEANS (eq 54); n_samples = number of multiples
 * of stress_every in (step, step+n_steps].  Returns n_samples. */
static int64_t run(const oracle_params *p, oracle_state *st, int64_t n_steps, double shear_rate,
                   const double *kappa, int64_t chains_per_group,
                   int stress_every, double *stress_out, int sample_every, oracle_corr *corr,
                   double guard, int n_threads)
{
    const int64_t M = p->n_chains;
    int64_t n_samples = 0;
    if (stress_every > 0) n_samples = (st->step + n_steps) / stress_every - st->step / stress_every;
    if (n_threads < 1) n_threads = 1;
    if ((int64_t)n_threads > M) n_threads = (int)M;
    work_t *w = (work_t *)calloc((size_t)n_threads, sizeof(work_t));
    pthread_t *th = (pthread_t *)calloc((size_t)n_threads, sizeof(pthread_t));
    /* Correlator sums are shared by the chains of a group: each thread adds into PRIVATE copies of
     * the sum / count arrays (rings and pending pairs are per chain, hence disjoint), merged below
     * in thread order, so that a multi-threaded run has no race and is reproducible. */
    const size_t nsum = corr ? (size_t)corr->groups * corr->levels * corr->bins : 0;
    oracle_corr *priv = corr && n_threads > 1 ? (oracle_corr *)calloc((size_t)n_threads, sizeof(oracle_corr)) : NULL;
    for (int t = 0; t < n_threads; ++t) {
        w[t].p = p; w[t].st = st; w[t].k0 = M * t / n_threads; w[t].k1 = M * (t + 1) / n_threads;
        w[t].n_steps = n_steps; w[t].shear_rate = shear_rate; w[t].stress_every = stress_every;
        w[t].stress_sum = n_samples ? (double *)calloc((size_t)n_samples * 12, sizeof(double)) : NULL;
        w[t].sample_every = sample_every; w[t].corr = corr; w[t].guard = guard;
        w[t].kappa = kappa; w[t].chains_per_group = chains_per_group;
        if (priv) {
            priv[t] = *corr;
            priv[t].sum = (double *)calloc(nsum, sizeof(double));
            priv[t].sum_gg = (double *)calloc(nsum, sizeof(double));
            priv[t].count = (int64_t *)calloc(nsum, sizeof(int64_t));
            w[t].corr = &priv[t];
        }
    }
    if (n_threads == 1) worker(&w[0]);
    else {
        for (int t = 0; t < n_threads; ++t) pthread_create(&th[t], NULL, worker, &w[t]);
        for (int t = 0; t < n_threads; ++t) pthread_join(th[t], NULL);
    }
    for (int64_t i = 0; i < n_samples * 12; ++i) {
        double s = 0.0;
        for (int t = 0; t < n_threads; ++t) s += w[t].stress_sum[i];
        stress_out[i] = s / (double)M;
    }
    if (priv) {
        for (int t = 0; t < n_threads; ++t) {
            for (size_t i = 0; i < nsum; ++i) {
                corr->sum[i] += priv[t].sum[i]; corr->sum_gg[i] += priv[t].sum_gg[i]; corr->count[i] += priv[t].count[i];
            }
            free(priv[t].sum); free(priv[t].sum_gg); free(priv[t].count);
        }
        free(priv);
    }
    for (int t = 0; t < n_threads; ++t) free(w[t].stress_sum);
    free(w); free(th);
    st->step += n_steps;
    return n_samples;
}

int64_t oracle_run(const oracle_params *p, oracle_state *st, int64_t n_steps, double shear_rate,
                   int stress_every, double *stress_out, int sample_every, oracle_corr *corr,
                   double guard, int n_threads)
{
    return run(p, st, n_steps, shear_rate, NULL, 1, stress_every, stress_out, sample_every, corr, guard, n_threads);
}

/* As oracle_run, with one velocity gradient tensor per block of chains_per_group consecutive local chains
 * (eqs 18, 21; the embedding of P:L17): kappa [ceil(M / chains_per_group)][9], row-major kappa_ab. */
int64_t oracle_run_kappa(const oracle_params *p, oracle_state *st, int64_t n_steps, int64_t chains_per_group,
                         const double *kappa, int stress_every, double *stress_out, int sample_every,
                         oracle_corr *corr, double guard, int n_threads)
{
    if (chains_per_group < 1 || !kappa) return -1;
    return run(p, st, n_steps, 0.0, kappa, chains_per_group, stress_every, stress_out, sample_every, corr, guard, n_threads);
}
