/*
 * tbsma_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU oracle for the TB-SMA (Cleri-Rosato form) Au force path of
 * arXiv:1311.3890 (French et al.).  Written from the paper text only; shares no code,
 * header, table or helper with the CUDA path under paper_1311_3890_b200/csrc/.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this library.
 *
 * Citations: "P:NN" = /root/reference/PAPER.md line NN.  "D:Ak" = reading Ak in DESIGN.md
 * (the places where the paper is silent, ambiguous or garbled).
 *
 * What is the plain definition (the method reaches it exactly, up to rounding order):
 *   rho_i = sum_{j != i, r_ij < r_cut} xi^2 exp(-2q (r_ij/r0 - 1))          P:47 Eq.1
 *   E_i   = sum_j A exp(-p (r_ij/r0 - 1)) - sqrt(rho_i)                      P:47-55 Eq.1-3
 *   E_C   = sum_i E_i                                                        P:55 Eq.3
 *   F_i   = -dE_C/dr_i  ("Differentiating eq 1 yields an expression for force that
 *           depends on the electron density rho of atoms i and j"; the explicit
 *           formula is derived in DESIGN.md and pinned by finite differences)
 *   W_ab  = 1/2 sum_i sum_j d_ij,a f_ij,b   (potential part of Eq.5; D:A11)
 * The functions below are brute force O(N^2) per replica: every ordered pair is tested.
 * A second, independent cell-list path (orc_compute_celllist) exists only so that the
 * full-size workloads can be checked in seconds; it is itself checked against the brute
 * force in tests/.
 *
 * Pins (tests/test_oracle_pins.py): dimer closed form, FCC lattice sums, F = -grad E by
 * central differences, momentum/torque conservation, rigid-motion invariance, virial
 * identities, OU closed form, NVE drift, cuRAND host Philox4x32-10.  No function here is
 * "parity unpinned" except that the paper's own printed physics (Table 3) is out of reach
 * (needs 10^6-step runs), as DESIGN.md states.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -fPIC -shared (see oracle/build.py).
 * -ffp-contract=off matters: the fp32 membership predicate (D:A6) is defined with an
 * explicit fmaf order and must not be re-contracted by the compiler.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_KB 8.617333262e-5    /* eV/K, CODATA (paper silent; D:units) */
#define ORC_ACC 9.648533212e-3   /* 1 eV/(A amu) expressed in A/fs^2 (D:units) */

typedef struct {
    double A, xi, p, q, r0, mass_amu; /* Table 1; r0 read as a/sqrt2 (D:A1) */
} orc_params;

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------
 * D:A6 -- membership predicate, DEFINED in fp32 so that an fp32 GPU and this oracle agree
 * bit for bit on which pairs exist:
 *   dx = x_i - x_j (fp32, round to nearest); on a periodic axis
 *        if (dx > L/2) dx -= L; else if (dx < -L/2) dx += L;   L = fl32(hi - lo)
 *   d2 = fmaf(dz,dz, fmaf(dy,dy, dx*dx));  include iff d2 < rmax*rmax (fp32 product),
 *   rmax = (float)(radius in double).
 * ---------------------------------------------------------------------------------- */
static inline int orc_member_f32(const float *pi, const float *pj, const float *L,
                                 const uint8_t *per, float r2max)
{
    float dx = pi[0] - pj[0];
    float dy = pi[1] - pj[1];
    float dz = pi[2] - pj[2];
    if (per[0]) { float h = 0.5f * L[0]; if (dx > h) dx -= L[0]; else if (dx < -h) dx += L[0]; }
    if (per[1]) { float h = 0.5f * L[1]; if (dy > h) dy -= L[1]; else if (dy < -h) dy += L[1]; }
    if (per[2]) { float h = 0.5f * L[2]; if (dz > h) dz -= L[2]; else if (dz < -h) dz += L[2]; }
    float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    return d2 < r2max;
}

/* fp64 displacement d = r_i - r_j with the minimum image on periodic axes (D:A7). */
static inline void orc_disp_f64(const double *xi, const double *xj, const double *L,
                                const uint8_t *per, double d[3])
{
    for (int a = 0; a < 3; ++a) {
        double t = xi[a] - xj[a];
        if (per[a]) { double h = 0.5 * L[a]; if (t > h) t -= L[a]; else if (t < -h) t += L[a]; }
        d[a] = t;
    }
}

/* Does the pair (i,j) interact inside radius r?  fp32_pred = 1: D:A6 on the float-cast
 * positions; fp32_pred = 0: the same test in double (for fp64-input invariance pins). */
static inline int orc_pair(const double *x, int64_t i, int64_t j, const float *Lf,
                           const double *Ld, const uint8_t *per, double r, int fp32_pred)
{
    if (fp32_pred) {
        float pi[3] = {(float)x[3 * i], (float)x[3 * i + 1], (float)x[3 * i + 2]};
        float pj[3] = {(float)x[3 * j], (float)x[3 * j + 1], (float)x[3 * j + 2]};
        float rf = (float)r;
        return orc_member_f32(pi, pj, Lf, per, rf * rf);
    }
    double d[3];
    orc_disp_f64(x + 3 * i, x + 3 * j, Ld, per, d);
    return d[0] * d[0] + d[1] * d[1] + d[2] * d[2] < r * r;
}

static void orc_box_len(const float *lo, const float *hi, int r, float Lf[3], double Ld[3])
{
    for (int a = 0; a < 3; ++a) {
        Lf[a] = hi[3 * r + a] - lo[3 * r + a]; /* fp32 difference: THE box length (D:A6) */
        Ld[a] = (double)Lf[a];
    }
}

/* ------------------------------------------------------------------------------------
 * Neighbour sets (D:A6, "neighbor list buffer radius").  Brute force: every ordered
 * pair of the replica.  pos4 = n x (x,y,z,w) floats.  list is n x max_nb, ascending j
 * (global index).  Returns the largest count found (may exceed max_nb: then lists are
 * truncated and the caller must treat it as an error), or -1 on bad arguments.
 * ---------------------------------------------------------------------------------- */
int orc_neighbors(int64_t n, const float *pos4, int32_t R, const int32_t *off,
                  const float *lo, const float *hi, const uint8_t *per, double radius,
                  int32_t max_nb, int32_t *counts, int32_t *list)
{
    if (n < 0 || R < 0 || max_nb < 0) return -1;
    int maxc = 0;
    float rf = (float)radius;
    float r2 = rf * rf;
    for (int32_t r = 0; r < R; ++r) {
        float Lf[3]; double Ld[3];
        orc_box_len(lo, hi, r, Lf, Ld);
        const uint8_t *pr = per + 3 * r;
#pragma omp parallel for schedule(dynamic, 64) reduction(max : maxc)
        for (int64_t i = off[r]; i < off[r + 1]; ++i) {
            int c = 0;
            for (int64_t j = off[r]; j < off[r + 1]; ++j) {
                if (j == i) continue;
                if (orc_member_f32(pos4 + 4 * i, pos4 + 4 * j, Lf, pr, r2)) {
                    if (c < max_nb) list[i * (int64_t)max_nb + c] = (int32_t)j;
                    ++c;
                }
            }
            counts[i] = c;
            if (c > maxc) maxc = c;
        }
    }
    return maxc;
}

/* ------------------------------------------------------------------------------------
 * Pair functions.  x_ij = r_ij/r0 - 1.
 *   phi_rho(r) = xi^2 exp(-2 q x)                      P:47 Eq.1 (summand)
 *   phi_rep(r) = A exp(-p x)                           P:51 Eq.2 (summand)
 * dE_C/dr_ij for the unordered pair {i,j}, s = rho^(-1/2):
 *   dE/dr = -(2 A p / r0) exp(-p x) + (q xi^2 / r0) exp(-2 q x) (s_i + s_j)
 * (the 2 on the repulsive term: Eq.2-3 count the pair from both ends, no 1/2, D:A3).
 * ---------------------------------------------------------------------------------- */
static inline double orc_phi_rho(const orc_params *P, double r)
{
    return P->xi * P->xi * exp(-2.0 * P->q * (r / P->r0 - 1.0));
}
static inline double orc_phi_rep(const orc_params *P, double r)
{
    return P->A * exp(-P->p * (r / P->r0 - 1.0));
}

/* Stage 1: rho_i for atoms [i0,i1) of one replica, brute force over the replica. */
static void orc_density_range(const orc_params *P, double r_cut, const double *x,
                              int64_t a0, int64_t a1, int64_t i0, int64_t i1,
                              const float *Lf, const double *Ld, const uint8_t *per,
                              int fp32_pred, double *rho)
{
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = i0; i < i1; ++i) {
        double s = 0.0;
        for (int64_t j = a0; j < a1; ++j) {
            if (j == i || !orc_pair(x, i, j, Lf, Ld, per, r_cut, fp32_pred)) continue;
            double d[3];
            orc_disp_f64(x + 3 * i, x + 3 * j, Ld, per, d);
            s += orc_phi_rho(P, sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
        }
        rho[i] = s;
    }
}

/* ------------------------------------------------------------------------------------
 * Full force/energy/virial evaluation, brute force (two stages as in P:59).
 *   x      n x 3 doubles (fp32 inputs promoted exactly when fp32_pred = 1)
 *   off    R+1 replica offsets; lo/hi R x 3 floats; per R x 3 bytes
 * Outputs (any may be NULL except rho): rho[n], e_atom[n], f[n*3], e_rep[R],
 *   w_rep[R*6] order xx yy zz xy xz yz.
 * ---------------------------------------------------------------------------------- */
int orc_compute(const orc_params *P, double r_cut, int64_t n, const double *x, int32_t R,
                const int32_t *off, const float *lo, const float *hi, const uint8_t *per,
                int fp32_pred, double *rho, double *e_atom, double *f, double *e_rep,
                double *w_rep)
{
    if (!P || !x || !rho || n < 0) return -1;
    for (int32_t r = 0; r < R; ++r) {
        float Lf[3]; double Ld[3];
        orc_box_len(lo, hi, r, Lf, Ld);
        const uint8_t *pr = per + 3 * r;
        const int64_t a0 = off[r], a1 = off[r + 1];
        /* stage 1: densities of every atom of the replica must be complete first */
        orc_density_range(P, r_cut, x, a0, a1, a0, a1, Lf, Ld, pr, fp32_pred, rho);
        /* stage 2 */
        double E = 0.0, W0 = 0, W1 = 0, W2 = 0, W3 = 0, W4 = 0, W5 = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : E, W0, W1, W2, W3, W4, W5)
        for (int64_t i = a0; i < a1; ++i) {
            double si = rho[i] > 0.0 ? 1.0 / sqrt(rho[i]) : 0.0; /* D:A5 */
            double erep = 0.0, fi[3] = {0, 0, 0};
            for (int64_t j = a0; j < a1; ++j) {
                if (j == i || !orc_pair(x, i, j, Lf, Ld, pr, r_cut, fp32_pred)) continue;
                double d[3];
                orc_disp_f64(x + 3 * i, x + 3 * j, Ld, pr, d);
                double rij = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                double sj = rho[j] > 0.0 ? 1.0 / sqrt(rho[j]) : 0.0;
                erep += orc_phi_rep(P, rij);
                double dEdr = -(2.0 * P->p / P->r0) * orc_phi_rep(P, rij) +
                              (P->q / P->r0) * orc_phi_rho(P, rij) * (si + sj);
                double fij[3]; /* force on i from j */
                for (int a = 0; a < 3; ++a) { fij[a] = -dEdr * d[a] / rij; fi[a] += fij[a]; }
                W0 += 0.5 * d[0] * fij[0]; W1 += 0.5 * d[1] * fij[1]; W2 += 0.5 * d[2] * fij[2];
                W3 += 0.5 * d[0] * fij[1]; W4 += 0.5 * d[0] * fij[2]; W5 += 0.5 * d[1] * fij[2];
            }
            double ei = erep - sqrt(rho[i]);
            if (e_atom) e_atom[i] = ei;
            if (f) { f[3 * i] = fi[0]; f[3 * i + 1] = fi[1]; f[3 * i + 2] = fi[2]; }
            E += ei;
        }
        if (e_rep) e_rep[r] = E;
        if (w_rep) {
            double *w = w_rep + 6 * r;
            w[0] = W0; w[1] = W1; w[2] = W2; w[3] = W3; w[4] = W4; w[5] = W5;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------
 * The same quantities for a SAMPLE of atoms, each computed one by one from scratch
 * (its own rho and the rho of each of its partners by brute force over the replica).
 * Used for parity at full workload sizes.  idx[m] global atom indices; rep_of[m] the
 * replica of each.  Outputs rho[m], e_atom[m], f[m*3].
 * ---------------------------------------------------------------------------------- */
int orc_compute_sample(const orc_params *P, double r_cut, const double *x, const int32_t *off,
                       const float *lo, const float *hi, const uint8_t *per, int fp32_pred,
                       int64_t m, const int64_t *idx, const int32_t *rep_of, double *rho,
                       double *e_atom, double *f)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < m; ++k) {
        const int64_t i = idx[k];
        const int32_t r = rep_of[k];
        float Lf[3]; double Ld[3];
        orc_box_len(lo, hi, r, Lf, Ld);
        const uint8_t *pr = per + 3 * r;
        const int64_t a0 = off[r], a1 = off[r + 1];
        double rho_i = 0.0;
        for (int64_t j = a0; j < a1; ++j) {
            if (j == i || !orc_pair(x, i, j, Lf, Ld, pr, r_cut, fp32_pred)) continue;
            double d[3];
            orc_disp_f64(x + 3 * i, x + 3 * j, Ld, pr, d);
            rho_i += orc_phi_rho(P, sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
        }
        double si = rho_i > 0.0 ? 1.0 / sqrt(rho_i) : 0.0;
        double erep = 0.0, fi[3] = {0, 0, 0};
        for (int64_t j = a0; j < a1; ++j) {
            if (j == i || !orc_pair(x, i, j, Lf, Ld, pr, r_cut, fp32_pred)) continue;
            double d[3];
            orc_disp_f64(x + 3 * i, x + 3 * j, Ld, pr, d);
            double rij = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            double rho_j = 0.0; /* partner's density, from scratch */
            for (int64_t l = a0; l < a1; ++l) {
                if (l == j || !orc_pair(x, j, l, Lf, Ld, pr, r_cut, fp32_pred)) continue;
                double e[3];
                orc_disp_f64(x + 3 * j, x + 3 * l, Ld, pr, e);
                rho_j += orc_phi_rho(P, sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]));
            }
            double sj = rho_j > 0.0 ? 1.0 / sqrt(rho_j) : 0.0;
            erep += orc_phi_rep(P, rij);
            double dEdr = -(2.0 * P->p / P->r0) * orc_phi_rep(P, rij) +
                          (P->q / P->r0) * orc_phi_rho(P, rij) * (si + sj);
            for (int a = 0; a < 3; ++a) fi[a] += -dEdr * d[a] / rij;
        }
        rho[k] = rho_i;
        if (e_atom) e_atom[k] = erep - sqrt(rho_i);
        if (f) { f[3 * k] = fi[0]; f[3 * k + 1] = fi[1]; f[3 * k + 2] = fi[2]; }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Philox4x32-10 counter-based generator (Salmon, Moraes, Dror, Shaw, SC'11), restated:
 * ten rounds of  (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
 * the key bumped by the Weyl constants between rounds (D:A9).  Pinned against cuRAND's
 * host generator CURAND_RNG_PSEUDO_PHILOX4_32_10 in tests/.
 * ---------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* D:A9 -- three standard normals for (replica seed, tag within replica, step):
 *   key = (seed_lo, seed_hi); counter = (tag, step_lo, step_hi, 0);
 *   u_k = ((x_k >> 8) + 0.5) 2^-24 in (0,1);
 *   (g0,g1) = sqrt(-2 ln u0) (cos 2 pi u1, sin 2 pi u1);  g2 = sqrt(-2 ln u2) cos 2 pi u3. */
void orc_gauss3(uint64_t seed, uint32_t tag, uint64_t step, double g[3], uint32_t raw[4])
{
    uint32_t ctr[4] = {tag, (uint32_t)step, (uint32_t)(step >> 32), 0u};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t o[4];
    orc_philox4x32_10(ctr, key, o);
    double u[4];
    for (int k = 0; k < 4; ++k) u[k] = ((double)(o[k] >> 8) + 0.5) * (1.0 / 16777216.0);
    const double twopi = 6.283185307179586476925286766559;
    double ra = sqrt(-2.0 * log(u[0])), rb = sqrt(-2.0 * log(u[2]));
    g[0] = ra * cos(twopi * u[1]);
    g[1] = ra * sin(twopi * u[1]);
    g[2] = rb * cos(twopi * u[3]);
    if (raw) { raw[0] = o[0]; raw[1] = o[1]; raw[2] = o[2]; raw[3] = o[3]; }
}

int orc_compute_celllist(const orc_params *P, double r_cut, int64_t n, const double *x, int32_t R,
                         const int32_t *off, const float *lo, const float *hi, const uint8_t *per,
                         int fp32_pred, double *rho, double *e_atom, double *f, double *e_rep,
                         double *w_rep, int64_t *n_pairs_directed);

/* ------------------------------------------------------------------------------------
 * One MD step ("integrated using the velocity Verlet algorithm with a time step of
 * 2.0 fs"; rigid gripping layers; thermostat per D:A8 = BAOAB Langevin, which is exactly
 * velocity Verlet when gamma = 0):
 *   B: v += (dt/2) (c/m) F        A: x += (dt/2) v
 *   O: v <- c1 v + c2 sigma_v g,  c1 = exp(-gamma dt), c2 = sqrt(1-c1^2),
 *      sigma_v = sqrt(kB T c / m), g ~ N(0,1)^3 from orc_gauss3(seed_r, tag, step)
 *   A: x += (dt/2) v              new F(x)          B: v += (dt/2) (c/m) F
 * Grip atoms (D:A12): flag 1 = fixed, flag 2 = pulled; v = 0; fixed atoms stay where they
 * are; a pulled atom is PLACED at z = zref + D_r (D_r = total slab displacement, D:A10).
 * On entry f must hold F(x); on exit x, v, f are those of the next step.  The tag of atom
 * i is i - off[r] (the oracle never reorders atoms).  ekin_rep: sum over dynamic atoms of
 * (m/2c) v^2 in eV after the final B.
 * ---------------------------------------------------------------------------------- */
int orc_md_step(const orc_params *P, double r_cut, int64_t n, double *x, double *v, double *f,
                const int32_t *flags, const double *zref, int32_t R, const int32_t *off,
                const float *lo, const float *hi, const uint8_t *per, int fp32_pred,
                double dt, const double *T, double gamma, const uint64_t *seed, uint64_t step,
                const double *slab_disp, int use_cells, double *rho, double *e_atom,
                double *e_rep, double *w_rep, double *ekin_rep)
{
    const double kick = 0.5 * dt * ORC_ACC / P->mass_amu;
    const double c1 = exp(-gamma * dt);
    const double c2 = sqrt(1.0 - c1 * c1);
    for (int32_t r = 0; r < R; ++r) {
        const double sigv = sqrt(ORC_KB * T[r] * ORC_ACC / P->mass_amu);
#pragma omp parallel for schedule(static)
        for (int64_t i = off[r]; i < off[r + 1]; ++i) {
            if (flags[i] == 0) {
                for (int a = 0; a < 3; ++a) v[3 * i + a] += kick * f[3 * i + a];      /* B */
                for (int a = 0; a < 3; ++a) x[3 * i + a] += 0.5 * dt * v[3 * i + a];  /* A */
                if (gamma > 0.0) {                                                    /* O */
                    double g[3];
                    orc_gauss3(seed[r], (uint32_t)(i - off[r]), step, g, NULL);
                    for (int a = 0; a < 3; ++a) v[3 * i + a] = c1 * v[3 * i + a] + c2 * sigv * g[a];
                }
                for (int a = 0; a < 3; ++a) x[3 * i + a] += 0.5 * dt * v[3 * i + a];  /* A */
            } else {
                v[3 * i] = v[3 * i + 1] = v[3 * i + 2] = 0.0;
                if (flags[i] == 2) x[3 * i + 2] = zref[i] + slab_disp[r];
            }
        }
    }
    /* use_cells = 1 swaps in the linked-cell evaluation of the same sums (for long runs) */
    int rc = use_cells ? orc_compute_celllist(P, r_cut, n, x, R, off, lo, hi, per, fp32_pred, rho,
                                              e_atom, f, e_rep, w_rep, NULL)
                       : orc_compute(P, r_cut, n, x, R, off, lo, hi, per, fp32_pred, rho, e_atom,
                                     f, e_rep, w_rep);
    if (rc) return rc;
    for (int32_t r = 0; r < R; ++r) {
        double ek = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : ek)
        for (int64_t i = off[r]; i < off[r + 1]; ++i) {
            if (flags[i] != 0) continue;
            for (int a = 0; a < 3; ++a) v[3 * i + a] += kick * f[3 * i + a];          /* B */
            ek += 0.5 * P->mass_amu / ORC_ACC *
                  (v[3 * i] * v[3 * i] + v[3 * i + 1] * v[3 * i + 1] + v[3 * i + 2] * v[3 * i + 2]);
        }
        if (ekin_rep) ekin_rep[r] = ek;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Second, independent CPU path: linked cells + the same pair formulas.  Exists so that
 * full-size workloads (10^6 atoms) can be checked and timed; validated against
 * orc_compute on <= 10 k atoms in tests/.  Cells are >= r_cut wide; an atom outside a
 * non-periodic box is clamped into the edge cell (still correct: an edge cell is
 * open-ended).  Periodic axes need >= 3 cells.
 * ---------------------------------------------------------------------------------- */
typedef struct {
    int nc[3]; double lo[3], w[3]; uint8_t per[3];
    int64_t a0, a1; int32_t *head; /* ncell+1 starts */ int32_t *items;
} orc_cells;

static int orc_cell_coord(const orc_cells *C, int a, double xa)
{
    int c = (int)floor((xa - C->lo[a]) / C->w[a]);
    if (C->per[a]) { c %= C->nc[a]; if (c < 0) c += C->nc[a]; }
    else { if (c < 0) c = 0; if (c >= C->nc[a]) c = C->nc[a] - 1; }
    return c;
}

static int orc_cells_build(orc_cells *C, const double *x, int64_t a0, int64_t a1,
                           const float *lo, const float *hi, const uint8_t *per, double rc)
{
    C->a0 = a0; C->a1 = a1;
    for (int a = 0; a < 3; ++a) {
        C->per[a] = per[a];
        double l = lo[a], h = hi[a];
        if (!per[a]) { /* bounding box of the atoms, so the caller's box need not be tight */
            double mn = 1e300, mx = -1e300;
            for (int64_t i = a0; i < a1; ++i) { double t = x[3 * i + a]; if (t < mn) mn = t; if (t > mx) mx = t; }
            if (a1 > a0) { l = mn; h = mx + 1e-9; }
        }
        int nc = (int)floor((h - l) / (rc * 1.000001));
        if (nc < 1) nc = 1;
        if (per[a] && nc < 3) return -2;
        C->nc[a] = nc; C->lo[a] = l; C->w[a] = (h - l) / nc;
    }
    int64_t ncell = (int64_t)C->nc[0] * C->nc[1] * C->nc[2];
    C->head = (int32_t *)calloc((size_t)ncell + 1, sizeof(int32_t));
    C->items = (int32_t *)malloc((size_t)(a1 - a0 > 0 ? a1 - a0 : 1) * sizeof(int32_t));
    if (!C->head || !C->items) return -3;
    int32_t *cid = (int32_t *)malloc((size_t)(a1 - a0 > 0 ? a1 - a0 : 1) * sizeof(int32_t));
    for (int64_t i = a0; i < a1; ++i) {
        int cx = orc_cell_coord(C, 0, x[3 * i]), cy = orc_cell_coord(C, 1, x[3 * i + 1]),
            cz = orc_cell_coord(C, 2, x[3 * i + 2]);
        int32_t c = (int32_t)(((int64_t)cz * C->nc[1] + cy) * C->nc[0] + cx);
        cid[i - a0] = c; C->head[c + 1]++;
    }
    for (int64_t c = 0; c < ncell; ++c) C->head[c + 1] += C->head[c];
    int32_t *fill = (int32_t *)calloc((size_t)ncell, sizeof(int32_t));
    for (int64_t i = a0; i < a1; ++i) { int32_t c = cid[i - a0]; C->items[C->head[c] + fill[c]++] = (int32_t)i; }
    free(fill); free(cid);
    return 0;
}

/* visit every j != i in the (up to) 27 cells around atom i that passes the predicate */
#define ORC_FOR_NEIGH(C, x, i, BODY)                                                         \
    {                                                                                        \
        int cc[3];                                                                           \
        for (int a = 0; a < 3; ++a) cc[a] = orc_cell_coord((C), a, (x)[3 * (i) + a]);        \
        for (int oz = -1; oz <= 1; ++oz) for (int oy = -1; oy <= 1; ++oy) for (int ox = -1; ox <= 1; ++ox) { \
            int c3[3] = {cc[0] + ox, cc[1] + oy, cc[2] + oz}; int ok = 1;                    \
            for (int a = 0; a < 3; ++a) {                                                    \
                if ((C)->per[a]) c3[a] = (c3[a] + (C)->nc[a]) % (C)->nc[a];                  \
                else if (c3[a] < 0 || c3[a] >= (C)->nc[a]) ok = 0;                           \
            }                                                                                \
            if (!ok) continue;                                                               \
            int64_t c = ((int64_t)c3[2] * (C)->nc[1] + c3[1]) * (C)->nc[0] + c3[0];          \
            for (int32_t t = (C)->head[c]; t < (C)->head[c + 1]; ++t) {                      \
                int64_t j = (C)->items[t];                                                   \
                if (j == (i)) continue;                                                      \
                BODY                                                                         \
            }                                                                                \
        }                                                                                    \
    }

int orc_compute_celllist(const orc_params *P, double r_cut, int64_t n, const double *x, int32_t R,
                         const int32_t *off, const float *lo, const float *hi, const uint8_t *per,
                         int fp32_pred, double *rho, double *e_atom, double *f, double *e_rep,
                         double *w_rep, int64_t *n_pairs_directed)
{
    if (!P || !x || !rho || n < 0) return -1;
    int64_t npairs = 0;
    for (int32_t r = 0; r < R; ++r) {
        float Lf[3]; double Ld[3];
        orc_box_len(lo, hi, r, Lf, Ld);
        const uint8_t *pr = per + 3 * r;
        orc_cells C;
        int rc = orc_cells_build(&C, x, off[r], off[r + 1], lo + 3 * r, hi + 3 * r, pr, r_cut);
        if (rc) return rc;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : npairs)
        for (int64_t i = off[r]; i < off[r + 1]; ++i) {
            double s = 0.0;
            ORC_FOR_NEIGH(&C, x, i, {
                if (orc_pair(x, i, j, Lf, Ld, pr, r_cut, fp32_pred)) {
                    double d[3];
                    orc_disp_f64(x + 3 * i, x + 3 * j, Ld, pr, d);
                    s += orc_phi_rho(P, sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
                    ++npairs;
                }
            })
            rho[i] = s;
        }
        double E = 0.0, W0 = 0, W1 = 0, W2 = 0, W3 = 0, W4 = 0, W5 = 0;
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : E, W0, W1, W2, W3, W4, W5)
        for (int64_t i = off[r]; i < off[r + 1]; ++i) {
            double si = rho[i] > 0.0 ? 1.0 / sqrt(rho[i]) : 0.0;
            double erep = 0.0, fi[3] = {0, 0, 0};
            ORC_FOR_NEIGH(&C, x, i, {
                if (orc_pair(x, i, j, Lf, Ld, pr, r_cut, fp32_pred)) {
                    double d[3];
                    orc_disp_f64(x + 3 * i, x + 3 * j, Ld, pr, d);
                    double rij = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                    double sj = rho[j] > 0.0 ? 1.0 / sqrt(rho[j]) : 0.0;
                    erep += orc_phi_rep(P, rij);
                    double dEdr = -(2.0 * P->p / P->r0) * orc_phi_rep(P, rij) +
                                  (P->q / P->r0) * orc_phi_rho(P, rij) * (si + sj);
                    double fij[3];
                    for (int a = 0; a < 3; ++a) { fij[a] = -dEdr * d[a] / rij; fi[a] += fij[a]; }
                    W0 += 0.5 * d[0] * fij[0]; W1 += 0.5 * d[1] * fij[1]; W2 += 0.5 * d[2] * fij[2];
                    W3 += 0.5 * d[0] * fij[1]; W4 += 0.5 * d[0] * fij[2]; W5 += 0.5 * d[1] * fij[2];
                }
            })
            double ei = erep - sqrt(rho[i]);
            if (e_atom) e_atom[i] = ei;
            if (f) { f[3 * i] = fi[0]; f[3 * i + 1] = fi[1]; f[3 * i + 2] = fi[2]; }
            E += ei;
        }
        if (e_rep) e_rep[r] = E;
        if (w_rep) {
            double *w = w_rep + 6 * r;
            w[0] = W0; w[1] = W1; w[2] = W2; w[3] = W3; w[4] = W4; w[5] = W5;
        }
        free(C.head); free(C.items);
    }
    if (n_pairs_directed) *n_pairs_directed = npairs;
    return 0;
}
