/*
 * rms_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-walker-at-a-time fp64 CPU oracle of the hot path of the
 * Realistic Microstructure Simulator (arXiv 2012.06478): the Monte Carlo random
 * walk through a 3d voxelised label lattice with elastic reflection / permeation,
 * PGSE phase, T2 weight and the final signal / moment sums.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference
 * legs may call this.  It shares no code, header, table or constant generator
 * with the CUDA path under paper_2012_06478_b200/csrc; the two only agree on
 * the counter scheme of the random numbers.
 *
 * Citations: "P:<n>" is a line of /root/reference/PAPER.md, with the section /
 * equation it falls in.  "R<n>" is a numbered reading in DESIGN.md (where the
 * paper is silent).
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"):
 *   philox4x32_10        known-answer vectors (tests/golden/philox4x32_10_kat.txt)
 *   direction            <u>=0, <u_k^2>=1/3, <u_k^4>=1/5, |u|=1, z<->-z symmetry
 *   tables               ds=0.049 um, Eq.3 = Eq.2a/(1+alpha),
 *                        P12/P21 = sqrt(D2/D1)
 *   step                 brute-force sub-stepped ray march on tiny random lattices,
 *                        all reflect/pass outcomes forced
 *   run, free            <X^2>=2Dt exactly in expectation, K=-6/(5N), S=prod sinc
 *   run, plates          closed-form narrow-pulse S(q,t) and <X^2>(t)
 *   run, equilibrium     uniform density kept with D contrast and permeable walls
 *                        (P:78), exchange between slabs vs. the eigen-series
 *   run, T2              alpha = exp(-t/T2) exactly for a single compartment (Eq.5)
 *   run, cylinder        short-time Mitra law D(t)/D0 = 1 - 4/(3 sqrt(pi)) (S_x/V) sqrt(D0 t)
 *                        with S_x/V counted on the staircase surface of the lattice cylinder
 *   run, encounters      membrane encounters per step = surface * step / 4
 *   run, absorbing walls surviving fraction between plates = Brownstein-Tarr series (Eq.4; R = rho S/V)
 *   run, T1 / mixing time alpha = exp(-(t_T2/T2 + t_mix/T1)) exactly per impermeable compartment (Eq.5);
 *                        T1 = T2 reproduces the run without a mixing time; well-mixed permeable slabs:
 *                        1 - <alpha> = f_b t_mix / T1_b to first order, for either starting compartment
 *   tables, conc         equal c = Eq.3 bit for bit; P_12/P_21 = c_2 sqrt(D_2) / (c_1 sqrt(D_1)); the chain Eq.C.9-C.13-C.14;
 *                        Eq.C.15 for kappa = inf
 *   run, conc            initial density ~ c_L; kept by permeable membranes with D contrast; barrier-limited exchange
 *                        rate k = 2 kappa (r^lambda / a_1 + r^(lambda-1) / a_2) between slabs
 *   tensor_signal (rms_oracle.py)  waveform on one axis rotated onto n = scalar waveform along n (same walkers, 1e-12);
 *                        free walk: <e^{-i phi}> = prod_k sinc(c ds |W_k|), W_k the vector suffix sums of g
 *   run, label_weight    label counts ~ w_L V_L; w_L = 1/V_L: equal walkers per cell, and the volume-weighted sum of the
 *                        per-cell signals (volume_weighted_signal, rms_oracle.py) = the uniform-density signal
 *   run, ERL             between plates: density (1 + h/ds)/2 within ds of a wall (Eq.A.1), gap narrowed by ds/8 per side
 *                        (Eq.A.8), D_parallel = D0 (1 + S/V ds / 16) (Eq.A.9)
 *   run, rejection sampl. D_parallel = D0 (1 - 3/16 S/V ds) between plates (Eq.B.2), uniform density
 * Parity unpinned: wide-pulse signals inside voxelised cylinders / axons have
 *   no closed form; they are pinned only through the pieces above.
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_OK 0
#define ORC_ERR_ARG -1
#define ORC_ERR_STEP_TOO_LARGE -2
#define ORC_ERR_P_RANGE -3
#define ORC_ERR_NO_SPACE -4
#define ORC_ERR_OOM -5

#define ORC_MAX_INIT_ATTEMPTS (1u << 20)

/* ------------------------------------------------------------------------- */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  R2: the paper names no  */
/* generator; north_star fixes this one, keyed on (seed, walker, step).        */
/* ------------------------------------------------------------------------- */
void rms_oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0; /* hi0:lo0 */
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2; /* hi1:lo1 */
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Counter layout (R2): key = (seed_lo, seed_hi); ctr = (walker_lo, walker_hi, index, stream). */
enum { STREAM_INIT = 0, STREAM_DIR = 1, STREAM_PERM = 2, STREAM_INIT_OFFSET = 3, STREAM_MT = 4, STREAM_ERL = 5 };
#define ORC_MAX_ERL_ATTEMPTS 4096u /* R25 */

static void draw(uint64_t seed, uint64_t walker, uint32_t index, uint32_t stream, uint32_t out[4])
{
    uint32_t ctr[4] = { (uint32_t)walker, (uint32_t)(walker >> 32), index, stream };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    rms_oracle_philox4x32_10(ctr, key, out);
}

/* R3: words -> reals, all exactly representable in fp32 as well as fp64.
 * sym(w) = (2*(w>>9) + 1 - 2^23) * 2^-23  in (-1,1), symmetric, never 0 or +-1.
 * uni(w) = (w>>8) * 2^-24                 in [0,1). */
static double sym(uint32_t w) { return ((double)(2 * (int64_t)(w >> 9) + 1 - 8388608)) / 8388608.0; }
static double uni(uint32_t w) { return (double)(w >> 8) / 16777216.0; }

/* R4 ("random direction in 3d"): z uniform in (-1,1), azimuth psi = pi*sym(wb)
 * (Archimedes' hat-box theorem => uniform on the sphere). */
void rms_oracle_direction(uint32_t wa, uint32_t wb, double u[3])
{
    const double pi = 3.14159265358979323846;
    double z = sym(wa);
    double psi = pi * sym(wb);
    double rho = sqrt(1.0 - z * z);
    u[0] = rho * cos(psi);
    u[1] = rho * sin(psi);
    u[2] = z;
}

/* Direction words of absolute 1-based step i (R2): one Philox call serves two steps. */
static void direction_words(uint64_t seed, uint64_t walker, int64_t step, uint32_t* wa, uint32_t* wb)
{
    uint32_t w[4];
    draw(seed, walker, (uint32_t)((step - 1) >> 1), STREAM_DIR, w);
    if (step & 1) { *wa = w[0]; *wb = w[1]; } else { *wa = w[2]; *wb = w[3]; }
}

/* Permeation uniforms of step i (R5): 33-bit uniforms u_e = (c_e + uni(v_e)) / 512 for the
 * e-th unlike-label encounter of the step, e = 0,1,2.  The 9 coarse bits c_0, c_1 are the
 * low 9 bits of the step's two direction words (unused by sym); c_2 = v_3 & 511.
 * v_0..v_3 = Philox(walker, index = step, stream PERM). */
static void permeation_uniforms(uint64_t seed, uint64_t walker, int64_t step, uint32_t wa, uint32_t wb, double u[3])
{
    uint32_t v[4];
    draw(seed, walker, (uint32_t)step, STREAM_PERM, v);
    u[0] = ((double)(wa & 511u) + uni(v[0])) / 512.0;
    u[1] = ((double)(wb & 511u) + uni(v[1])) / 512.0;
    u[2] = ((double)(v[3] & 511u) + uni(v[2])) / 512.0;
}

/* Saturation (magnetisation transfer) uniforms of step i (R20): u_e = uni(m_e) for the e-th
 * unlike-label encounter of the step, m_0..m_3 = Philox(walker, index = step, stream MT). */
static void saturation_uniforms(uint64_t seed, uint64_t walker, int64_t step, double u[3])
{
    uint32_t m[4];
    draw(seed, walker, (uint32_t)step, STREAM_MT, m);
    u[0] = uni(m[0]); u[1] = uni(m[1]); u[2] = uni(m[2]);
}

/* Absorbing membranes / surface relaxation (Eq.4): a walker in label a that meets a
 * membrane towards label b is saturated with probability P_MT = rho_ab ds_a / D_a C_d, the
 * same C_d as in Eq.2a.  Rounded once to an fp32-representable value (R6). */
int rms_oracle_mt_table(int n_labels, const float* D, const float* rho, double dt_ms, double* Q_out)
{
    const double C3 = 2.0 / 3.0;
    if (n_labels <= 0 || !D || !rho || !(dt_ms > 0)) return ORC_ERR_ARG;
    for (int a = 0; a < n_labels; ++a)
        for (int b = 0; b < n_labels; ++b) {
            double q = 0.0;
            if (a != b) {
                double r = (double)rho[a * n_labels + b];
                if (r < 0 || r != r) return ORC_ERR_ARG;
                q = r * sqrt(6.0 * dt_ms / (double)D[a]) * C3;
                if (q > 1.0) return ORC_ERR_P_RANGE;
            }
            Q_out[a * n_labels + b] = (double)(float)q;
        }
    return ORC_OK;
}

/* ------------------------------------------------------------------------- */
/* Tables (Eq.1, Eq.2-3, P:678-681 Eq.C.15).                    */
/* s[L]  = sqrt(6 D_L dt) / l_p : hop length in voxel units (d = 3).           */
/* P[a][b] permeation probability from label a into label b.                   */
/* Both are rounded once to fp32-representable values (R6).                    */
/* ------------------------------------------------------------------------- */
int rms_oracle_tables_conc(int n_labels, const float* D, const float* kappa, const float* conc, double voxel_um,
                           double dt_ms, double* s_out, double* P_out);

int rms_oracle_tables(int n_labels, const float* D, const float* kappa, double voxel_um, double dt_ms,
                      double* s_out, double* P_out)
{
    return rms_oracle_tables_conc(n_labels, D, kappa, NULL, voxel_um, dt_ms, s_out, P_out);
}

/* The same with a spin concentration c_L per label (Appendix C.2, Eq.C.9, C.13-C.14; Appendix C.3, Eq.C.15):
 *   P_ab = A_ab r^lambda / (1 + alpha),  alpha = (A_ab r^lambda + A_ba r^(lambda-1)) / 2,  r = c_b / c_a,
 *   lambda = 1 / (1 + c_b sqrt(D_b) / (c_a sqrt(D_a)))   (the paper's arg min of alpha_lambda; R24)
 * which is Eq.C.9 with kappa_0 = kappa (1 - alpha) of Eq.C.13, and Eq.3 for r = 1.  conc = NULL: all equal. */
int rms_oracle_tables_conc(int n_labels, const float* D, const float* kappa, const float* conc, double voxel_um,
                           double dt_ms, double* s_out, double* P_out)
{
    const double C3 = 2.0 / 3.0; /* Eq.2b, d = 3 */
    if (n_labels <= 0 || !D || !(voxel_um > 0) || !(dt_ms > 0)) return ORC_ERR_ARG;
    for (int a = 0; a < n_labels; ++a) {
        if (!(D[a] > 0)) return ORC_ERR_ARG;
        double s = sqrt(6.0 * (double)D[a] * dt_ms) / voxel_um; /* Eq.1 */
        s_out[a] = (double)(float)s;
        if (!(s_out[a] < 1.0)) return ORC_ERR_STEP_TOO_LARGE;   /* ds < l_p */
    }
    if (!P_out) return ORC_OK;
    for (int a = 0; a < n_labels; ++a) {
        for (int b = 0; b < n_labels; ++b) {
            double P;
            if (a == b) {
                P = 1.0;
            } else {
                double k = kappa ? (double)kappa[a * n_labels + b] : 0.0;
                double Da = D[a], Db = D[b];
                double ca = conc ? (double)conc[a] : 1.0, cb = conc ? (double)conc[b] : 1.0;
                if (k < 0 || k != k) return ORC_ERR_ARG;
                if (!(ca >= 0) || !(cb >= 0) || isinf(ca) || isinf(cb)) return ORC_ERR_ARG;
                if (k == 0.0 || ca == 0.0 || cb == 0.0) {
                    P = 0.0; /* impermeable; nothing enters (or sits in) a medium without spins */
                } else if (isinf(k)) {
                    /* no membrane between media of different D and c: Eq.C.15 */
                    P = cb * sqrt(Db) / (ca * sqrt(Da));
                    if (P > 1.0) P = 1.0;
                } else if (ca != cb) {
                    double r = cb / ca;
                    double lam = 1.0 / (1.0 + cb * sqrt(Db) / (ca * sqrt(Da)));
                    double Aab = k * sqrt(6.0 * dt_ms / Da) * C3 * pow(r, lam);       /* Eq.C.9a */
                    double Aba = k * sqrt(6.0 * dt_ms / Db) * C3 * pow(r, lam - 1.0); /* Eq.C.9b */
                    P = Aab / (1.0 + 0.5 * (Aab + Aba));                              /* Eq.C.13-C.14 */
                    if (P > 1.0) return ORC_ERR_P_RANGE;
                } else {
                    double Aab = k * sqrt(6.0 * dt_ms / Da) * C3; /* kappa ds_a / D_a C_d, Eq.2a */
                    double Aba = k * sqrt(6.0 * dt_ms / Db) * C3;
                    P = Aab / (1.0 + 0.5 * (Aab + Aba));          /* Eq.3 */
                    if (P > 1.0) return ORC_ERR_P_RANGE;          /* R9 */
                }
            }
            P_out[a * n_labels + b] = (double)(float)P;
        }
    }
    return ORC_OK;
}

/* ------------------------------------------------------------------------- */
/* One Monte Carlo step (P:152-159 steps 2-4; Fig.2).         */
/* Coordinates in voxel units: unwrapped voxel vox[3], offset off[3] in [0,1). */
/* u[3] unit direction, up[3] permeation uniforms for encounters 0,1,2.        */
/* ------------------------------------------------------------------------- */
typedef struct {
    int nx, ny, nz;
    const uint16_t* labels;
    int n_labels;
    const double* s; /* [n_labels] */
    const double* P; /* [n_labels^2] */
    const double* Q; /* [n_labels^2] saturation probability P_MT, or NULL (no absorbing membranes) */
    int rejection;   /* 1: rejection sampling (Appendix B), 2: equal-step-length random leap (Appendix A) */
} lattice_t;

static int wrap(int64_t a, int n) { int64_t m = a % n; return (int)(m < 0 ? m + n : m); }

static uint16_t label_at(const lattice_t* lat, const int32_t v[3])
{
    int x = wrap(v[0], lat->nx), y = wrap(v[1], lat->ny), z = wrap(v[2], lat->nz); /* R1: periodic box */
    return lat->labels[((size_t)z * lat->ny + y) * lat->nx + x];
}

/* permeation uniforms are drawn only when a membrane with 0 < P < 1 is met (same values either way) */
typedef struct { uint64_t seed, walker; int64_t step; uint32_t wa, wb; int have; double u[3]; } perm_src_t;

static double perm_uniform(perm_src_t* ps, int e)
{
    if (!ps->have) { permeation_uniforms(ps->seed, ps->walker, ps->step, ps->wa, ps->wb, ps->u); ps->have = 1; }
    return ps->u[e < 3 ? e : 2];
}

/* saturation uniforms, drawn only when an absorbing membrane (P_MT > 0) is met */
typedef struct { uint64_t seed, walker; int64_t step; int have; double u[3]; } mt_src_t;

static double mt_uniform(mt_src_t* ms, int e)
{
    if (!ms->have) { saturation_uniforms(ms->seed, ms->walker, ms->step, ms->u); ms->have = 1; }
    return ms->u[e < 3 ? e : 2];
}

static void step_core(const lattice_t* lat, int32_t vox[3], double off[3], uint16_t* label,
                      const double u[3], perm_src_t* ps, mt_src_t* ms, int* saturated,
                      int* n_enc, int* n_perm, int* n_clamp, int* cancelled)
{
    if (cancelled) *cancelled = 0;
    uint16_t L = *label;
    const uint16_t L_in = L;
    const int32_t v_in[3] = { vox[0], vox[1], vox[2] };
    const int n_perm_in = *n_perm;
    double r[3], p[3];
    int done[3] = { 0, 0, 0 };
    int e = 0;
    for (int k = 0; k < 3; ++k) { r[k] = lat->s[L] * u[k]; p[k] = off[k]; } /* R8: ds of the label at the start */

    for (int it = 0; it < 3; ++it) { /* at most three interactions */
        int kstar = -1;
        double tmin = 0.0;
        for (int k = 0; k < 3; ++k) {
            if (done[k]) continue;
            double g = p[k] + r[k];
            if (g >= 1.0 || g < 0.0) {
                double t = ((r[k] > 0.0 ? 1.0 : 0.0) - p[k]) / r[k];
                if (kstar < 0 || t < tmin) { kstar = k; tmin = t; } /* R10: ties -> lowest axis */
            }
        }
        if (kstar < 0) break;
        int sigma = r[kstar] > 0.0 ? 1 : -1;
        for (int k = 0; k < 3; ++k) { p[k] += tmin * r[k]; r[k] *= (1.0 - tmin); }
        p[kstar] = sigma > 0 ? 1.0 : 0.0; /* exactly on the face */

        int32_t nb[3] = { vox[0], vox[1], vox[2] };
        nb[kstar] += sigma;
        uint16_t Ln = label_at(lat, nb);
        int pass;
        if (Ln == L) {
            pass = 1; /* face between voxels of one compartment is no membrane */
        } else {
            double P = lat->P[(size_t)L * lat->n_labels + Ln];
            ++*n_enc;
            if (lat->Q && ms) { /* Eq.4: the encounter saturates the walker with probability P_MT; its walk goes on */
                double Q = lat->Q[(size_t)L * lat->n_labels + Ln];
                if (Q > 0.0 && mt_uniform(ms, e) < Q) *saturated = 1;
            }
            pass = (P >= 1.0) || (P > 0.0 && perm_uniform(ps, e) < P); /* permeate with probability P */
            ++e;
            if (pass) ++*n_perm;
        }
        if (pass) {
            vox[kstar] += sigma;
            p[kstar] = sigma > 0 ? 0.0 : 1.0;
            if (Ln != L) {
                double scale = lat->s[Ln] / lat->s[L]; /* R7: rest of dt is spent at the new speed */
                for (int k = 0; k < 3; ++k) r[k] *= scale;
                L = Ln;
            }
        } else if (lat->rejection) {
            /* rejection sampling (Appendix B): a step that meets a membrane it does not cross is cancelled and
             * the walker does not move for the step */
            vox[0] = v_in[0]; vox[1] = v_in[1]; vox[2] = v_in[2];
            *label = L_in;
            *n_perm = n_perm_in; /* a permeation earlier in the cancelled step did not happen either */
            if (cancelled) *cancelled = 1;
            return;
        } else {
            r[kstar] = -r[kstar]; /* elastic collision on the face plane */
        }
        done[kstar] = 1;
    }
    for (int k = 0; k < 3; ++k) {
        double f = p[k] + r[k];
        const double fmax = 1.0 - 1.0 / 9007199254740992.0; /* 1 - 2^-53 */
        if (f < 0.0) { f = 0.0; ++*n_clamp; }
        if (f > fmax) { f = fmax; ++*n_clamp; }
        off[k] = f;
    }
    *label = L;
}

/* Exported single step, for the brute-force pins.  s[n_labels], P[n_labels^2] given directly. */
int rms_oracle_step(int nx, int ny, int nz, const uint16_t* labels, int n_labels, const double* s, const double* P,
                    int32_t vox[3], double off[3], uint16_t* label, const double u[3], const double up[3],
                    int32_t counts[3])
{
    lattice_t lat = { nx, ny, nz, labels, n_labels, s, P, NULL, 0 };
    int ne = 0, np = 0, nc = 0;
    perm_src_t ps = { 0, 0, 0, 0, 0, 1, { up[0], up[1], up[2] } };
    step_core(&lat, vox, off, label, u, &ps, NULL, NULL, &ne, &np, &nc, NULL);
    counts[0] = ne; counts[1] = np; counts[2] = nc;
    return ORC_OK;
}

/* Walker initialisation (P:151 step 1; R13): rejection sampling of a uniform voxel until its label
 * is allowed, then a uniform in-voxel offset.  Integer arithmetic: v = floor(uni(w) * n). */
int rms_oracle_init_walker_conc(int nx, int ny, int nz, const uint16_t* labels, const uint8_t* label_allowed,
                                const float* accept, uint64_t seed, uint64_t walker, int32_t vox[3], double off[3],
                                uint16_t* label);

int rms_oracle_init_walker(int nx, int ny, int nz, const uint16_t* labels, const uint8_t* label_allowed,
                           uint64_t seed, uint64_t walker, int32_t vox[3], double off[3], uint16_t* label)
{
    return rms_oracle_init_walker_conc(nx, ny, nz, labels, label_allowed, NULL, seed, walker, vox, off, label);
}

/* With spin concentrations the equilibrium density is proportional to c_L (Appendix C.2): a proposed voxel is kept
 * with probability accept[L] = c_L / max c over the allowed labels, drawn from the spare fourth word (R24). */
int rms_oracle_init_walker_conc(int nx, int ny, int nz, const uint16_t* labels, const uint8_t* label_allowed,
                                const float* accept, uint64_t seed, uint64_t walker, int32_t vox[3], double off[3],
                                uint16_t* label)
{
    uint32_t w[4];
    for (uint32_t a = 0; a < ORC_MAX_INIT_ATTEMPTS; ++a) {
        draw(seed, walker, a, STREAM_INIT, w);
        int x = (int)(((uint64_t)(w[0] >> 8) * (uint64_t)nx) >> 24);
        int y = (int)(((uint64_t)(w[1] >> 8) * (uint64_t)ny) >> 24);
        int z = (int)(((uint64_t)(w[2] >> 8) * (uint64_t)nz) >> 24);
        uint16_t L = labels[((size_t)z * ny + y) * nx + x];
        if (label_allowed && !label_allowed[L]) continue;
        if (accept && !(uni(w[3]) < (double)accept[L])) continue;
        vox[0] = x; vox[1] = y; vox[2] = z;
        *label = L;
        draw(seed, walker, 0, STREAM_INIT_OFFSET, w);
        off[0] = uni(w[0]); off[1] = uni(w[1]); off[2] = uni(w[2]);
        return ORC_OK;
    }
    return ORC_ERR_NO_SPACE;
}

/* ------------------------------------------------------------------------- */
/* Whole run: init -> n_steps steps -> sums (Eq.5, Eq.7).           */
/* ------------------------------------------------------------------------- */
typedef struct {
    /* substrate */
    lattice_t lat;
    double voxel_um;
    const double* inv_T2; /* [n_labels], 0 = no relaxation */
    const double* inv_T1; /* [n_labels], 0 = no relaxation; used in the mixing time */
    int64_t mix_first, mix_steps; /* steps mix_first .. mix_first + mix_steps - 1 (1-based) are the mixing time */
    const uint16_t* label_class;
    int n_classes;
    /* walkers */
    uint64_t n_walkers, first_id, seed;
    const uint8_t* label_allowed;
    const float* accept; /* [n_labels] c_L / max c, or NULL (spin concentrations, R24) */
    /* run */
    double dt;
    int64_t n_steps;
    int n_wave; const float* wave;
    int n_g; const double* gamp;
    int n_dir; const double* dirs;
    int n_snap; const int64_t* snap_steps;
    /* per-walker outputs (optional) */
    int32_t* final_vox; double* final_off; uint16_t* final_label;
    int32_t* init_vox; double* init_off; double* phi; double* relax;
} job_t;

typedef struct {
    const job_t* job;
    uint64_t w_begin, w_end; /* indices into [0, n_walkers) */
    double *sum_alpha, *sig_re, *sig_im, *m2, *m4, *snap_alpha;
    uint64_t* class_flow;
    uint64_t counters[5];
    int status;
} part_t;

static size_t n_sig(const job_t* j) { return (size_t)j->n_wave * j->n_g * j->n_dir * j->n_classes; }
static size_t n_mom(const job_t* j) { return (size_t)j->n_snap * j->n_dir * j->n_classes; }
static size_t n_sal(const job_t* j) { return (size_t)j->n_snap * j->n_classes; }
static size_t n_flow(const job_t* j) { return (size_t)j->n_snap * j->n_classes * j->n_classes; }

static void* run_part(void* arg)
{
    part_t* pt = (part_t*)arg;
    const job_t* j = pt->job;
    const lattice_t* lat = &j->lat;
    double* Phi = (double*)malloc(sizeof(double) * 3 * (size_t)(j->n_wave > 0 ? j->n_wave : 1));
    if (!Phi) { pt->status = ORC_ERR_OOM; return NULL; }

    for (uint64_t wi = pt->w_begin; wi < pt->w_end; ++wi) {
        uint64_t id = j->first_id + wi;
        int32_t v0[3], v[3];
        double f0[3], f[3];
        uint16_t L0, L;
        int st = rms_oracle_init_walker_conc(lat->nx, lat->ny, lat->nz, lat->labels, j->label_allowed, j->accept, j->seed, id, v0,
                                              f0, &L0);
        if (st != ORC_OK) { pt->status = st; break; }
        memcpy(v, v0, sizeof v); memcpy(f, f0, sizeof f); L = L0;
        int c0 = j->label_class ? j->label_class[L0] : 0;
        double R = 0.0; /* sum_i t_i / T2^(i), Eq.5 */
        for (int m = 0; m < 3 * j->n_wave; ++m) Phi[m] = 0.0;
        int snap = 0;

        for (int64_t i = 1; i <= j->n_steps; ++i) {
            uint32_t wa, wb;
            double u[3];
            int ne = 0, np = 0, nc = 0;
            direction_words(j->seed, id, i, &wa, &wb);
            rms_oracle_direction(wa, wb, u);
            perm_src_t ps = { j->seed, id, i, wa, wb, 0, { 0, 0, 0 } };
            mt_src_t ms = { j->seed, id, i, 0, { 0, 0, 0 } };
            int sat = 0;
            int cancelled = 0;
            step_core(lat, v, f, &L, u, &ps, &ms, &sat, &ne, &np, &nc, &cancelled);
            /* equal-step-length random leap (R25): a cancelled step is tried again in a new direction, drawn
             * from the stream ERL of this step and attempt, until it meets no membrane */
            for (uint32_t a = 1; lat->rejection == 2 && cancelled && a < ORC_MAX_ERL_ATTEMPTS; ++a) {
                uint32_t w4[4];
                draw(j->seed, id, (uint32_t)i, STREAM_ERL | (a << 8), w4);
                rms_oracle_direction(w4[0], w4[1], u);
                step_core(lat, v, f, &L, u, &ps, &ms, &sat, &ne, &np, &nc, &cancelled);
            }
            if (sat && !isinf(R)) { R = INFINITY; pt->counters[4] += 1; } /* Eq.4: alpha_rho = 0 from here on */
            pt->counters[0] += (uint64_t)ne; pt->counters[1] += (uint64_t)np; pt->counters[2] += (uint64_t)nc;
            if ((uint64_t)ne > pt->counters[3]) pt->counters[3] = (uint64_t)ne;

            /* displacement in voxel units; the integer part is exact */
            double dx[3];
            for (int k = 0; k < 3; ++k) dx[k] = (double)(v[k] - v0[k]) + (f[k] - f0[k]);
            /* Eq.7 phase, right-endpoint rule (R11): Phi_m += w_m[i] (x_i - x_0) */
            for (int m = 0; m < j->n_wave; ++m) {
                double w = (double)j->wave[(size_t)m * j->n_steps + (i - 1)];
                for (int k = 0; k < 3; ++k) Phi[3 * m + k] += w * dx[k];
            }
            /* Eq.5: whole dt to the compartment at the end of the hop (R12) */
            /* stimulated echo: during the mixing time the magnetisation is along B0 and Eq.5 runs with T1 (R22) */
            int mixing = i >= j->mix_first && i < j->mix_first + j->mix_steps;
            R += j->dt * (mixing ? j->inv_T1[L] : j->inv_T2[L]); /* (stays +inf once saturated) */

            while (snap < j->n_snap && j->snap_steps[snap] == i) {
                double alpha = exp(-R);
                int cn = j->label_class ? j->label_class[L] : 0;
                pt->snap_alpha[(size_t)snap * j->n_classes + c0] += alpha;
                pt->class_flow[((size_t)snap * j->n_classes + c0) * j->n_classes + cn] += 1;
                for (int d = 0; d < j->n_dir; ++d) {
                    const double* n = j->dirs + 3 * d;
                    double X = j->voxel_um * (n[0] * dx[0] + n[1] * dx[1] + n[2] * dx[2]);
                    size_t o = ((size_t)snap * j->n_dir + d) * j->n_classes + c0;
                    pt->m2[o] += alpha * X * X;
                    pt->m4[o] += alpha * X * X * X * X;
                }
                ++snap;
            }
        }
        /* signal sums, Eq.7: alpha e^{-i phi} */
        double alpha = exp(-R);
        pt->sum_alpha[c0] += alpha;
        for (int m = 0; m < j->n_wave; ++m)
            for (int g = 0; g < j->n_g; ++g)
                for (int d = 0; d < j->n_dir; ++d) {
                    const double* n = j->dirs + 3 * d;
                    double proj = n[0] * Phi[3 * m] + n[1] * Phi[3 * m + 1] + n[2] * Phi[3 * m + 2];
                    double ph = j->gamp[(size_t)m * j->n_g + g] * j->dt * j->voxel_um * proj;
                    size_t o = (((size_t)m * j->n_g + g) * j->n_dir + d) * j->n_classes + c0;
                    pt->sig_re[o] += alpha * cos(ph);
                    pt->sig_im[o] -= alpha * sin(ph);
                }
        if (j->final_vox) memcpy(j->final_vox + 3 * wi, v, sizeof v);
        if (j->final_off) memcpy(j->final_off + 3 * wi, f, sizeof f);
        if (j->final_label) j->final_label[wi] = L;
        if (j->init_vox) memcpy(j->init_vox + 3 * wi, v0, sizeof v0);
        if (j->init_off) memcpy(j->init_off + 3 * wi, f0, sizeof f0);
        if (j->phi) memcpy(j->phi + 3 * (size_t)j->n_wave * wi, Phi, sizeof(double) * 3 * (size_t)j->n_wave);
        if (j->relax) j->relax[wi] = R;
    }
    free(Phi);
    return NULL;
}

int rms_oracle_run(
    int nx, int ny, int nz, double voxel_um, const uint16_t* labels, int n_labels,
    const float* D, const float* T2, const float* kappa, const float* rho, const uint16_t* label_class, int n_classes,
    uint64_t n_walkers, uint64_t first_id, const uint8_t* label_allowed, uint64_t seed,
    double dt_ms, int64_t n_steps, int n_wave, const float* wave, int n_g, const double* gamp,
    int n_dir, const double* dirs, int n_snap, const int64_t* snap_steps, int n_threads, int interaction,
    const float* T1, int64_t mix_first, int64_t mix_steps, const float* conc, const float* label_weight,
    double* sum_alpha, double* sig_re, double* sig_im, double* m2, double* m4, double* snap_alpha,
    uint64_t* class_flow, uint64_t* counters,
    int32_t* final_vox, double* final_off, uint16_t* final_label,
    int32_t* init_vox, double* init_off, double* phi, double* relax)
{
    if (nx <= 0 || ny <= 0 || nz <= 0 || !labels || n_labels <= 0 || n_classes <= 0 || n_steps < 0 ||
        n_wave < 0 || n_g < 0 || n_dir < 0 || n_snap < 0 || !sum_alpha || !counters)
        return ORC_ERR_ARG;
    size_t nvox = (size_t)nx * ny * nz;
    for (size_t i = 0; i < nvox; ++i) if (labels[i] >= n_labels) return ORC_ERR_ARG;
    if (label_class) for (int a = 0; a < n_labels; ++a) if (label_class[a] >= n_classes) return ORC_ERR_ARG;
    for (int s = 0; s < n_snap; ++s) {
        if (snap_steps[s] < 1 || snap_steps[s] > n_steps) return ORC_ERR_ARG;
        if (s > 0 && snap_steps[s] <= snap_steps[s - 1]) return ORC_ERR_ARG;
    }
    for (int d = 0; d < n_dir; ++d) {
        const double* n = dirs + 3 * d;
        if (fabs(n[0] * n[0] + n[1] * n[1] + n[2] * n[2] - 1.0) > 1e-6) return ORC_ERR_ARG;
    }

    double* s_tab = (double*)malloc(sizeof(double) * n_labels);
    double* P_tab = (double*)malloc(sizeof(double) * (size_t)n_labels * n_labels);
    double* inv_T2 = (double*)malloc(sizeof(double) * 2 * n_labels);
    double* inv_T1 = inv_T2 ? inv_T2 + n_labels : NULL;
    double* Q_tab = rho ? (double*)malloc(sizeof(double) * (size_t)n_labels * n_labels) : NULL;
    if (!s_tab || !P_tab || !inv_T2 || (rho && !Q_tab)) { free(s_tab); free(P_tab); free(inv_T2); free(Q_tab); return ORC_ERR_OOM; }
    int st = rms_oracle_tables_conc(n_labels, D, kappa, conc, voxel_um, dt_ms, s_tab, P_tab);
    float* accept = NULL;
    if (st == ORC_OK && (conc || label_weight)) {
        /* initial density proportional to c_L (R24) times the caller's placement weight of the label (walkers per
         * axon; R26), over the allowed labels */
        double wmax = 0.0;
        accept = (float*)malloc(sizeof(float) * n_labels);
        if (!accept) st = ORC_ERR_OOM;
        for (int a = 0; a < n_labels && st == ORC_OK; ++a) {
            double w = (conc ? (double)conc[a] : 1.0) * (label_weight ? (double)label_weight[a] : 1.0);
            if (!(w >= 0.0) || isinf(w)) st = ORC_ERR_ARG;
            if ((!label_allowed || label_allowed[a]) && w > wmax) wmax = w;
        }
        if (st == ORC_OK && !(wmax > 0.0)) st = ORC_ERR_NO_SPACE;
        for (int a = 0; a < n_labels && st == ORC_OK; ++a)
            accept[a] = (float)((conc ? (double)conc[a] : 1.0) * (label_weight ? (double)label_weight[a] : 1.0) / wmax);
        if (st == ORC_OK && conc && interaction == 1) st = ORC_ERR_ARG; /* Appendix B.1 has no concentrations */
    }
    if (st == ORC_OK && rho) st = rms_oracle_mt_table(n_labels, D, rho, dt_ms, Q_tab);
    if (st == ORC_OK && interaction == 1 && kappa) {
        /* rejection sampling has its own permeation probability: P_T / (1 - P_T) = kappa ds / D0 C_d (Appendix B.1,
         * generalised to 3d with Eq.2a); the paper derives it for equal diffusivities on both sides only */
        for (int a = 0; a < n_labels && st == ORC_OK; ++a)
            for (int b = 0; b < n_labels; ++b) {
                double k = (double)kappa[a * n_labels + b];
                if (a == b || k == 0.0 || isinf(k)) continue;
                if (D[a] != D[b]) { st = ORC_ERR_ARG; break; }
                double A = k * sqrt(6.0 * dt_ms / (double)D[a]) * (2.0 / 3.0);
                P_tab[a * n_labels + b] = (double)(float)(A / (1.0 + A));
            }
    }
    if (interaction < 0 || interaction > 2) st = ORC_ERR_ARG;
    if (st == ORC_OK && interaction == 2) {
        /* ERL is defined for impermeable, non-absorbing membranes: a face is a wall (P = 0) or no membrane (P = 1) */
        if (rho) st = ORC_ERR_ARG;
        for (int a = 0; a < n_labels * n_labels && st == ORC_OK; ++a)
            if (P_tab[a] > 0.0 && P_tab[a] < 1.0) st = ORC_ERR_ARG;
    }
    if (mix_steps < 0 || (mix_steps > 0 && (mix_first < 1 || mix_first + mix_steps - 1 > n_steps))) st = ORC_ERR_ARG;
    if (st != ORC_OK) { free(s_tab); free(P_tab); free(inv_T2); free(Q_tab); free(accept); return st; }
    for (int a = 0; a < n_labels; ++a) {
        double t2 = T2 ? (double)T2[a] : 0.0;
        inv_T2[a] = (t2 > 0.0 && !isinf(t2)) ? 1.0 / t2 : 0.0; /* T2 <= 0 or inf: no relaxation */
        double t1 = T1 ? (double)T1[a] : 0.0;
        inv_T1[a] = (t1 > 0.0 && !isinf(t1)) ? 1.0 / t1 : 0.0; /* likewise; T1 = NULL: no relaxation in the mixing time */
    }

    job_t job;
    memset(&job, 0, sizeof job);
    job.lat.nx = nx; job.lat.ny = ny; job.lat.nz = nz; job.lat.labels = labels; job.lat.n_labels = n_labels;
    job.lat.s = s_tab; job.lat.P = P_tab; job.lat.Q = Q_tab; job.lat.rejection = interaction; /* 0 elastic collision, 1 rejection sampling, 2 ERL */
    job.voxel_um = voxel_um; job.inv_T2 = inv_T2; job.inv_T1 = inv_T1; job.mix_first = mix_first; job.mix_steps = mix_steps; job.label_class = label_class; job.n_classes = n_classes;
    job.n_walkers = n_walkers; job.first_id = first_id; job.seed = seed; job.label_allowed = label_allowed; job.accept = accept;
    job.dt = dt_ms; job.n_steps = n_steps; job.n_wave = n_wave; job.wave = wave; job.n_g = n_g; job.gamp = gamp;
    job.n_dir = n_dir; job.dirs = dirs; job.n_snap = n_snap; job.snap_steps = snap_steps;
    job.final_vox = final_vox; job.final_off = final_off; job.final_label = final_label;
    job.init_vox = init_vox; job.init_off = init_off; job.phi = phi; job.relax = relax;

    if (n_threads < 1) n_threads = 1;
    if ((uint64_t)n_threads > n_walkers && n_walkers > 0) n_threads = (int)n_walkers;
    part_t* parts = (part_t*)calloc((size_t)n_threads, sizeof(part_t));
    pthread_t* tids = (pthread_t*)calloc((size_t)n_threads, sizeof(pthread_t));
    int status = ORC_OK;
    if (!parts || !tids) { status = ORC_ERR_OOM; goto done; }
    for (int t = 0; t < n_threads; ++t) {
        part_t* p = &parts[t];
        p->job = &job;
        p->w_begin = n_walkers * (uint64_t)t / (uint64_t)n_threads;
        p->w_end = n_walkers * (uint64_t)(t + 1) / (uint64_t)n_threads;
        p->sum_alpha = (double*)calloc((size_t)n_classes, sizeof(double));
        p->sig_re = (double*)calloc(n_sig(&job) + 1, sizeof(double));
        p->sig_im = (double*)calloc(n_sig(&job) + 1, sizeof(double));
        p->m2 = (double*)calloc(n_mom(&job) + 1, sizeof(double));
        p->m4 = (double*)calloc(n_mom(&job) + 1, sizeof(double));
        p->snap_alpha = (double*)calloc(n_sal(&job) + 1, sizeof(double));
        p->class_flow = (uint64_t*)calloc(n_flow(&job) + 1, sizeof(uint64_t));
        if (!p->sum_alpha || !p->sig_re || !p->sig_im || !p->m2 || !p->m4 || !p->snap_alpha || !p->class_flow)
            status = ORC_ERR_OOM;
    }
    if (status == ORC_OK) {
        /* walker ids are only partitioned over threads; every walker's arithmetic is unchanged */
        for (int t = 1; t < n_threads; ++t) pthread_create(&tids[t], NULL, run_part, &parts[t]);
        run_part(&parts[0]);
        for (int t = 1; t < n_threads; ++t) pthread_join(tids[t], NULL);
        for (int c = 0; c < n_classes; ++c) sum_alpha[c] = 0.0;
        if (sig_re) memset(sig_re, 0, sizeof(double) * n_sig(&job));
        if (sig_im) memset(sig_im, 0, sizeof(double) * n_sig(&job));
        if (m2) memset(m2, 0, sizeof(double) * n_mom(&job));
        if (m4) memset(m4, 0, sizeof(double) * n_mom(&job));
        if (snap_alpha) memset(snap_alpha, 0, sizeof(double) * n_sal(&job));
        if (class_flow) memset(class_flow, 0, sizeof(uint64_t) * n_flow(&job));
        memset(counters, 0, sizeof(uint64_t) * 5);
        for (int t = 0; t < n_threads; ++t) { /* partial sums added in walker order */
            part_t* p = &parts[t];
            if (p->status != ORC_OK) status = p->status;
            for (int c = 0; c < n_classes; ++c) sum_alpha[c] += p->sum_alpha[c];
            if (sig_re) for (size_t i = 0; i < n_sig(&job); ++i) sig_re[i] += p->sig_re[i];
            if (sig_im) for (size_t i = 0; i < n_sig(&job); ++i) sig_im[i] += p->sig_im[i];
            if (m2) for (size_t i = 0; i < n_mom(&job); ++i) m2[i] += p->m2[i];
            if (m4) for (size_t i = 0; i < n_mom(&job); ++i) m4[i] += p->m4[i];
            if (snap_alpha) for (size_t i = 0; i < n_sal(&job); ++i) snap_alpha[i] += p->snap_alpha[i];
            if (class_flow) for (size_t i = 0; i < n_flow(&job); ++i) class_flow[i] += p->class_flow[i];
            counters[0] += p->counters[0]; counters[1] += p->counters[1]; counters[2] += p->counters[2];
            if (p->counters[3] > counters[3]) counters[3] = p->counters[3];
            counters[4] += p->counters[4];
        }
    }
done:
    if (parts) for (int t = 0; t < n_threads; ++t) {
        free(parts[t].sum_alpha); free(parts[t].sig_re); free(parts[t].sig_im); free(parts[t].m2);
        free(parts[t].m4); free(parts[t].snap_alpha); free(parts[t].class_flow);
    }
    free(parts); free(tids); free(s_tab); free(P_tab); free(inv_T2); free(Q_tab); free(accept);
    return status;
}
