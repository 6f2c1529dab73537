/*
 * c8opt_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct fp64 CPU restatement of the hot path of
 * arxiv 2309.15861 (Baack & Alameddine, ICRC2023): track segment -> Cherenkov /
 * fluorescence photons -> straight-line propagation through an n(h) atmosphere
 * -> telescope-sphere intersection -> per-telescope tally / photon records.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, header, table or
 * constant generator with the CUDA path (paper_2309_15861_b200/csrc): the two
 * were written independently from the paper and from DESIGN.md's readings.
 *
 * Every function cites the passage it follows: "PAPER.md:<line>" is the paper
 * text, "R<n>" is a reading of a point on which the paper is silent, listed in
 * DESIGN.md §2 (they are SURVEY.md §8(c)'s readings).
 *
 * The method is a Monte-Carlo sampling procedure, so the oracle is the
 * algorithm itself, step by step, in the paper's order: no blocking, fusion or
 * reordering.  The random numbers are a counter-based generator
 * (Philox4x32-10, Salmon et al., SC'11) keyed by (seed, segment id, photon
 * index) so that an independent implementation draws the same stream.
 *
 * Pins (tests/test_oracle_pins.py): Philox known-answer vectors; Frank-Tamm
 * constant, Cherenkov angle, threshold and photons per metre; column depth;
 * optical delay of a vertical ray; rotation-matrix invariants; ray-sphere
 * against an independent quadratic solver; isotropic acceptance fraction;
 * beamed/isotropic equality of expectation; wavelength law; ring geometry;
 * transmission special cases; conservation laws.  End-to-end photon-level
 * results are "parity unpinned by the paper" (it prints no worked example);
 * they are pinned only through the above.
 *
 * Units: metres, nanoseconds, nanometres (wavelength), g/cm^2 (depth), MeV.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#define ORC_C_M_PER_NS 0.299792458           /* speed of light */
#define ORC_ALPHA      7.2973525693e-3       /* fine-structure constant (CODATA 2018) */
#define ORC_PI         3.14159265358979323846

typedef struct { double h_lo, a, b, c; } orc_layer; /* T(h) = a + b exp(-h/c) for h >= h_lo */

typedef struct {
    int n_layers;
    orc_layer layers[8];
    double eta0, rho0, h_obs;          /* n(h) - 1 = eta0 * rho(h) / rho0 ; rho0 in g/cm^3 */
    int tau_nh, tau_nl;                /* optical-depth table, 0 = none */
    double tau_h0, tau_dh, tau_l0, tau_dl;
    const float *tau;                  /* [nh][nl], row-major */
} orc_atmosphere;

typedef struct {
    uint64_t seed;
    uint32_t processes;                /* bit0 Cherenkov, bit1 fluorescence */
    double lam1, lam2, bunch_size;     /* Cherenkov band (nm), B */
    double fl_yield, fl_lam1, fl_lam2; /* photons / MeV, fluorescence band (nm) */
    int fl_beam_telescope;             /* -1 = isotropic */
    double fl_beam_halfangle;          /* rad */
    int refract;                       /* R27: apply the refraction corrections of PAPER.md:77 to position and angle */
    int cut_mode;                      /* R29: 0 none, 1 angle to the experiment centre, 2 smallest angle to a telescope */
    double cut_angle;                  /* rad ("recommended cut of 6 degrees") */
    double cauchy_b;                   /* R30: dispersion n(lambda, h) - 1 = eta(h) (1 + b / lambda^2), b in nm^2; 0 = none */
} orc_params;

/* one fp32 segment record, 12 x 4 bytes (flags is a uint32 in the same slot) */
typedef struct { float x0, y0, z0, t0, dx, dy, dz, length, gamma, charge, dE; uint32_t flags; } orc_segment;

/* everything that is constant over the photons of one (segment, process) */
typedef struct {
    uint32_t n_b;       /* number of photon bunches                                  */
    double mu;          /* expected photon number                                    */
    double w0;          /* weight per bunch                                          */
    double p0[3], d[3]; /* start point, unit direction                               */
    double L, t0, inv_beta_c;
    double sin_c, cos_c;/* Cherenkov angle (Cherenkov only)                          */
    double A[3];        /* bisecting vector of the rotation            */
    double M[3][3];     /* M_Rod                                       */
    double one_minus_cos_ab; /* beamed fluorescence: 1 - cos(alpha_b)                */
    int kind;           /* 0 Cherenkov, 1 fluorescence isotropic, 2 fluorescence beamed */
    double disp_eta, disp_beta2, disp_mean;  /* R30 (cauchy_b > 0): eta(h_mid), beta^2, band average of sin^2 theta_c */
} orc_frame;

typedef struct {
    double e[3], v[3];  /* emission point, unit direction */
    double t_e, lam, w; /* emission time (ns), wavelength (nm), weight before transmission */
} orc_photon;

typedef struct { uint64_t hits; double sum_w, sum_wt; } orc_tally;

/* one hit: x, y on the plane z = c_z relative to the centre; direction cosines; time; wavelength; weight */
typedef struct { double x, y, cx, cy, t, lam, w; uint64_t id; int32_t tel; int32_t pad; } orc_record;

/* ---------------------------------------------------------------------- */
/* Philox4x32-10, Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as
 * easy as 1, 2, 3", SC'11: multipliers 0xD2511F53 / 0xCD9E8D57, Weyl key
 * increments 0x9E3779B9 / 0xBB67AE85, 10 rounds.  (north_star: "counter-based
 * Philox4x32-10 keyed by (seed, segment id, photon index)"; R20.) */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
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

/* R19: U = ((r >> 9) + 1/2) * 2^-23, in (0,1), exactly representable in fp32 and fp64 */
double orc_uniform(uint32_t r)
{
    return ((double)(r >> 9) + 0.5) * (1.0 / 8388608.0);
}

/* ---------------------------------------------------------------------- */
/* Atmosphere (R18, SURVEY.md §8(c) "Atmosphere"): layer i is the last one with
 * h >= h_lo,i (layer 0 below the first boundary). */
static int orc_layer_of(const orc_atmosphere *atm, double h)
{
    int i = 0;
    for (int k = 1; k < atm->n_layers; ++k)
        if (h >= atm->layers[k].h_lo) i = k;
    return i;
}

/* column depth T(h) = a_i + b_i exp(-h / c_i)  [g/cm^2]  (BASELINE.json configs[1]) */
double orc_depth(const orc_atmosphere *atm, double h)
{
    const orc_layer *l = &atm->layers[orc_layer_of(atm, h)];
    return l->a + l->b * exp(-h / l->c);
}

/* density rho(h) = -dT/dh = (b_i / c_i) exp(-h / c_i)  [g/cm^2 per m] -> g/cm^3 by /100 */
double orc_density(const orc_atmosphere *atm, double h)
{
    const orc_layer *l = &atm->layers[orc_layer_of(atm, h)];
    return (l->b / l->c) * exp(-h / l->c) / 100.0;
}

/* refractivity eta(h) = n(h) - 1 = eta0 * rho(h) / rho0 */
double orc_refractivity(const orc_atmosphere *atm, double h)
{
    return atm->eta0 * orc_density(atm, h) / atm->rho0;
}

/* ---------------------------------------------------------------------- */
/* Rodrigues 180-degree matrix, printed entry by entry:
 *   M = 1 + 2 R^2 with A the bisecting vector between the flight direction and
 * the downward normal.  R6: A = normalize(dir - z^), fallback A = x^ when
 * 1 - dir_z < 1e-12. */
static void orc_rodrigues(const double dir[3], double A[3], double M[3][3])
{
    if (1.0 - dir[2] < 1e-12) {
        A[0] = 1.0; A[1] = 0.0; A[2] = 0.0;
    } else {
        double ax = dir[0], ay = dir[1], az = dir[2] - 1.0;
        double n = sqrt(ax * ax + ay * ay + az * az);
        A[0] = ax / n; A[1] = ay / n; A[2] = az / n;
    }
    double Ax = A[0], Ay = A[1], Az = A[2];
    M[0][0] = -2.0 * Ay * Ay - 2.0 * Az * Az + 1.0; M[0][1] = 2.0 * Ax * Ay; M[0][2] = 2.0 * Ax * Az;
    M[1][0] = 2.0 * Ax * Ay; M[1][1] = -2.0 * Ax * Ax - 2.0 * Az * Az + 1.0; M[1][2] = 2.0 * Ay * Az;
    M[2][0] = 2.0 * Ax * Az; M[2][1] = 2.0 * Ay * Az; M[2][2] = -2.0 * Ax * Ax - 2.0 * Ay * Ay + 1.0;
}

/* ---------------------------------------------------------------------- */
/* Per-(segment, process) preamble.  Returns 0 and fills *f; f->n_b = 0 when
 * no photon is emitted.  A segment with a non-finite field, gamma <= 1,
 * L < 0 or |d| off unity by more than 1e-3 is invalid: return -1, n_b = 0.
 *
 * tag 0, Cherenkov (R1-R3):
 *   eta = eta(z0 + L d_z / 2)                       (homogeneous step, midpoint)
 *   q = beta^2 n^2 - 1 = 2 eta + eta^2 - (1+eta)^2 / gamma^2   (cancellation-free)
 *   q <= 0  -> below threshold, Theta(beta - 1/n) = 0
 *   sin^2 theta_c = 1 - 1/(beta^2 n^2) = q / (beta^2 n^2)
 *   mu = 2 pi alpha z^2 L sin^2 theta_c (1/lam1 - 1/lam2)      (Frank-Tamm, mu_r = 1)
 *   n_b = ceil(mu / B), w0 = mu / n_b                          (R1)
 * tag 1, fluorescence (R13): mu = Y dE, same bunching;
 *   beamed (R14, R15): weight *= Omega / 4 pi, Omega = 2 pi (1 - cos alpha_b),
 *   line of sight from the segment midpoint to the telescope centre.
 */
/* R30: sin^2 theta_c at x = 1 / lambda [1/nm] for refractivity eta (long-wavelength value), beta^2, Cauchy coefficient b;
 * <= 0 below the threshold. */
double orc_dispersion_sin2(double eta, double beta2, double b, double x)
{
    double n = 1.0 + eta * (1.0 + (b * x) * x);
    double bn2 = (beta2 * n) * n;
    return 1.0 - 1.0 / bn2;
}

/* int_{x2}^{x1} max(0, sin^2 theta_c(x)) dx, composite Simpson, 16 intervals */
double orc_dispersion_integral(double eta, double beta2, double b, double x1, double x2)
{
    double h = (x1 - x2) / 16.0, odd = 0.0, even = 0.0, ends = 0.0;
    for (int k = 0; k <= 16; ++k) {
        double f = orc_dispersion_sin2(eta, beta2, b, x2 + (double)k * h);
        if (!(f > 0.0)) f = 0.0;
        if (k == 0 || k == 16) ends += f; else if (k & 1) odd += f; else even += f;
    }
    return (h / 3.0) * ((ends + 4.0 * odd) + 2.0 * even);
}

int orc_preamble(const orc_atmosphere *atm, const orc_params *par, const orc_segment *s, int tag,
                 const double *beam_tel_xyz, orc_frame *f)
{
    f->n_b = 0; f->mu = 0.0; f->w0 = 0.0;
    double L = (double)s->length, gamma = (double)s->gamma, zq = (double)s->charge;
    double dx = (double)s->dx, dy = (double)s->dy, dz = (double)s->dz;
    double dn = sqrt(dx * dx + dy * dy + dz * dz);
    if (!isfinite(s->x0) || !isfinite(s->y0) || !isfinite(s->z0) || !isfinite(s->t0) || !isfinite(dn) ||
        !isfinite(L) || !isfinite(gamma) || !isfinite(zq) || !isfinite(s->dE))
        return -1;
    if (!(gamma > 1.0) || !(L >= 0.0) || !(fabs(dn - 1.0) <= 1e-3))
        return -1;
    f->p0[0] = s->x0; f->p0[1] = s->y0; f->p0[2] = s->z0;
    f->d[0] = dx / dn; f->d[1] = dy / dn; f->d[2] = dz / dn;
    f->L = L; f->t0 = s->t0;
    double ig2 = 1.0 / (gamma * gamma);
    double beta = sqrt(1.0 - ig2);
    f->inv_beta_c = 1.0 / (beta * ORC_C_M_PER_NS);       /* R7: the particle moves at beta c */
    f->sin_c = 0.0; f->cos_c = 1.0; f->one_minus_cos_ab = 0.0;

    double mu;
    if (tag == 0) {
        f->kind = 0;
        double h_mid = f->p0[2] + 0.5 * L * f->d[2];      /* R3 */
        double eta = orc_refractivity(atm, h_mid);
        if (par->cauchy_b > 0.0) {
            /* R30: the Frank-Tamm integrand with n(lambda): in x = 1 / lambda,
             *   N = 2 pi alpha z^2 L int_{x2}^{x1} sin^2 theta_c(x) Theta(...) dx,  sin^2 theta_c(x) = 1 - 1 / (beta^2 n(x)^2),
             *   n(x) - 1 = eta (1 + b x^2)  (two-term Cauchy form; the paper gives no dispersion law),
             * by composite Simpson with 16 intervals; Theta cuts the integrand at 0 where beta n(x) < 1. */
            if (!(L > 0.0)) return 0;
            double S = orc_dispersion_integral(eta, 1.0 - ig2, par->cauchy_b, 1.0 / par->lam1, 1.0 / par->lam2);
            if (!(S > 0.0)) return 0;
            mu = 2.0 * ORC_PI * ORC_ALPHA * 1.0e9 * zq * zq * L * S;
            f->disp_eta = eta; f->disp_beta2 = 1.0 - ig2;
            f->disp_mean = S / (1.0 / par->lam1 - 1.0 / par->lam2);
            orc_rodrigues(f->d, f->A, f->M);
            goto bunches;
        }
        double q = 2.0 * eta + eta * eta - (1.0 + eta) * (1.0 + eta) * ig2;
        if (!(q > 0.0) || !(L > 0.0)) return 0;          /* threshold Theta(beta - 1/n) */
        double bn2 = (1.0 - ig2) * (1.0 + eta) * (1.0 + eta); /* beta^2 n^2 */
        double sin2 = q / bn2;
        f->cos_c = 1.0 / sqrt(bn2);                      /* cos theta_c = 1/(beta n) */
        f->sin_c = sqrt(sin2);
        double c_ft = 2.0 * ORC_PI * ORC_ALPHA * (1.0 / par->lam1 - 1.0 / par->lam2) * 1.0e9; /* per metre */
        mu = c_ft * zq * zq * L * sin2;
        orc_rodrigues(f->d, f->A, f->M);
        f->disp_eta = eta; f->disp_beta2 = 1.0 - ig2; f->disp_mean = sin2;
    } else {
        mu = par->fl_yield * (double)s->dE;               /* constant yield x total energy loss */
        if (par->fl_beam_telescope == -2) {
            /* R28 ("an opening angle and pointing depending on the telescope distance ... From the
             * resulting solid angle, the required scaling factor is calculated and applied to the total number of
             * photons ... for multiple telescopes, an emission area is defined which includes all telescopes"):
             * beam_tel_xyz = (centre, R_b) of a sphere that holds every telescope sphere.  Seen from the segment
             * midpoint m at distance D, every direction from any point of the track to any point of that sphere lies
             * within alpha of the line m -> centre, sin(alpha) = (R_b + L/2) / D.  The emission is uniform in that cone
             * and the NUMBER of photons is scaled by Omega / 4 pi = (1 - cos alpha) / 2 (weights stay mu'/n_b).
             * D <= R_b + L/2 (inside the array): isotropic, unscaled. */
            double u[3];
            for (int i = 0; i < 3; ++i) u[i] = beam_tel_xyz[i] - (f->p0[i] + (0.5 * L) * f->d[i]);
            double D = sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
            double sa = (beam_tel_xyz[3] + 0.5 * L) / D;
            if (sa < 1.0) {
                f->kind = 2;
                for (int i = 0; i < 3; ++i) u[i] /= D;
                orc_rodrigues(u, f->A, f->M);
                double ca = sqrt(1.0 - sa * sa);
                f->one_minus_cos_ab = (sa * sa) / (1.0 + ca);    /* 1 - cos(alpha) without cancellation */
                mu = mu * (0.5 * f->one_minus_cos_ab);
            } else {
                f->kind = 1;
            }
        } else if (par->fl_beam_telescope >= 0) {
            f->kind = 2;
            double los[3];
            for (int i = 0; i < 3; ++i) los[i] = beam_tel_xyz[i] - (f->p0[i] + 0.5 * L * f->d[i]);
            double ln = sqrt(los[0] * los[0] + los[1] * los[1] + los[2] * los[2]);
            for (int i = 0; i < 3; ++i) los[i] /= ln;
            orc_rodrigues(los, f->A, f->M);
            double sh = sin(0.5 * par->fl_beam_halfangle);
            f->one_minus_cos_ab = 2.0 * sh * sh;
        } else {
            f->kind = 1;
        }
    }
bunches:
    if (!(mu > 0.0)) return 0;
    double nb = ceil(mu / par->bunch_size);
    if (nb > 16777215.0) return -1;                      /* photon index must fit 24 bits of the record id */
    f->mu = mu;
    f->n_b = (uint32_t)nb;
    f->w0 = mu / nb;
    if (f->kind == 2 && par->fl_beam_telescope >= 0)
        f->w0 *= f->one_minus_cos_ab * 0.5;              /* R14 (weight form): Omega / 4 pi = (1 - cos alpha_b) / 2 */
    return 0;
}

/* ---------------------------------------------------------------------- */
/* Photon j of (segment S, process tag): R20 counter/key mapping, then
 * PAPER.md:49 (generate downward at the origin with the Cherenkov angle,
 * rotate the cone into the track direction, translate to the emission point),
 * PAPER.md:61 (photon vector), PAPER.md:69-71 (matrix). */
void orc_make_photon(const orc_frame *f, const orc_params *par, uint64_t S, uint32_t j, int tag, orc_photon *ph)
{
    /* R20: fluorescence (tag 1) draws one Philox block per photon, counter (j, S_lo, S_hi, 1), words -> u1..u4.
     * Cherenkov (tag 0) needs a position, an azimuth and a wavelength: one block, counter (j >> 1, S_lo, S_hi, 0),
     * serves the two photons 2k and 2k + 1: words (a, b) = (r0, r1) for the even one, (r2, r3) for the odd one;
     * u1 = U(a), u2 = U(b) from their upper 23 bits (R19), and the wavelength uniform from the 9 + 9 lower bits
     * those leave over: u3 = ((a & 511) 2^9 + (b & 511) + 1/2) 2^-18. */
    uint32_t ctr[4] = { tag == 0 ? (j >> 1) : j, (uint32_t)S, (uint32_t)(S >> 32), (uint32_t)tag };
    uint32_t key[2] = { (uint32_t)par->seed, (uint32_t)(par->seed >> 32) };
    uint32_t r[4];
    orc_philox4x32_10(ctr, key, r);
    double u1, u2, u3, u4;
    if (tag == 0) {
        uint32_t a = r[2 * (j & 1u)], b = r[2 * (j & 1u) + 1];
        u1 = orc_uniform(a); u2 = orc_uniform(b);
        u3 = ((double)(((a & 511u) << 9) | (b & 511u)) + 0.5) / 262144.0;
        u4 = 0.0;
    } else {
        u1 = orc_uniform(r[0]); u2 = orc_uniform(r[1]); u3 = orc_uniform(r[2]); u4 = orc_uniform(r[3]);
    }

    double s = u1 * f->L;                                  /* "randomly distributed along the track" PAPER.md:35 */
    for (int i = 0; i < 3; ++i) ph->e[i] = f->p0[i] + s * f->d[i];
    ph->t_e = f->t0 + s * f->inv_beta_c;                   /* R7 */
    ph->w = f->w0;

    double phi = 2.0 * ORC_PI * u2;                        /* R5: c_rng */
    double p[3];
    if (f->kind == 0) {
        double sin_c = f->sin_c, cos_c = f->cos_c;
        double x = 1.0 / par->lam1 - u3 * (1.0 / par->lam1 - 1.0 / par->lam2);
        if (par->cauchy_b > 0.0) {
            /* R30: the photon of wavelength 1 / x leaves at ITS Cherenkov angle, cos theta_c = 1 / (beta n(x)); x is still
             * drawn uniformly (R4), so the bunch carries sin^2 theta_c(x) / <sin^2 theta_c> as a weight factor (0 below
             * the threshold at this wavelength: the bunch is dropped by the caller) */
            double n = 1.0 + f->disp_eta * (1.0 + (par->cauchy_b * x) * x);
            double s2 = orc_dispersion_sin2(f->disp_eta, f->disp_beta2, par->cauchy_b, x);
            if (!(s2 > 0.0)) { ph->w = 0.0; s2 = 0.0; }
            else ph->w = f->w0 * (s2 / f->disp_mean);
            sin_c = sqrt(s2); cos_c = 1.0 / (sqrt(f->disp_beta2) * n);
        }
        p[0] = cos(phi) * sin_c; p[1] = sin(phi) * sin_c; p[2] = -cos_c;
        ph->lam = 1.0 / x;                                                /* R4: pdf ~ lambda^-2 */
    } else if (f->kind == 1) {
        double cth = 1.0 - 2.0 * u4, sth = 2.0 * sqrt(u4 * (1.0 - u4));            /* R16 isotropic */
        ph->v[0] = cos(phi) * sth; ph->v[1] = sin(phi) * sth; ph->v[2] = -cth;
        ph->lam = par->fl_lam1 + u3 * (par->fl_lam2 - par->fl_lam1);               /* R4 uniform */
        return;
    } else {
        double t = u4 * f->one_minus_cos_ab;               /* R14: uniform in the cone, 1 - cos theta' */
        double cth = 1.0 - t, sth = sqrt(t * (2.0 - t));
        p[0] = cos(phi) * sth; p[1] = sin(phi) * sth; p[2] = -cth;
        ph->lam = par->fl_lam1 + u3 * (par->fl_lam2 - par->fl_lam1);
    }
    for (int i = 0; i < 3; ++i)                             /* v = M_Rod p */
        ph->v[i] = f->M[i][0] * p[0] + f->M[i][1] * p[1] + f->M[i][2] * p[2];
}

/* ---------------------------------------------------------------------- */
/* R10: a hit is "distance from the sphere centre to the forward ray <= R":
 *   m = c - e ; s_c = m . v (closest approach along the ray) ; b^2 = |m|^2 - s_c^2
 *   hit <=> v_z < 0 and e_z > c_z and b^2 <= R^2 and s_c > 0.
 * Also returns the crossing of the horizontal plane through the centre (R11):
 *   s_pl = (c_z - e_z) / v_z ; (x, y) = e + s_pl v - c. */
int orc_intersect(const double e[3], const double v[3], const double tel[4],
                  double *b2, double *s_c, double *s_pl, double xy[2])
{
    double m[3] = { tel[0] - e[0], tel[1] - e[1], tel[2] - e[2] };
    double sc = m[0] * v[0] + m[1] * v[1] + m[2] * v[2];
    double bb = m[0] * m[0] + m[1] * m[1] + m[2] * m[2] - sc * sc;
    *b2 = bb; *s_c = sc;
    if (!(v[2] < 0.0) || !(e[2] > tel[2])) { *s_pl = 0.0; xy[0] = xy[1] = 0.0; return 0; }
    double sp = (tel[2] - e[2]) / v[2];
    *s_pl = sp;
    xy[0] = e[0] + sp * v[0] - tel[0];
    xy[1] = e[1] + sp * v[1] - tel[1];
    return (bb <= tel[3] * tel[3]) && (sc > 0.0);
}

/* R8: arrival time = emission time + optical path / c along the straight line
 * to the plane point: geometric length s_pl plus the excess integral of
 * eta dl = (eta0 / rho0) * (T(c_z) - T(e_z)) / |v_z|   [cm] -> x 0.01 [m]. */
double orc_arrival_time(const orc_atmosphere *atm, double e_z, double c_z, double v_z, double s_pl, double t_e)
{
    double excess_m = 0.01 * (atm->eta0 / atm->rho0) * (orc_depth(atm, c_z) - orc_depth(atm, e_z)) / fabs(v_z);
    return t_e + (s_pl + excess_m) / ORC_C_M_PER_NS;
}

/* R27 ("straight line propagation followed by the application of correction factors which changes
 * the arrival angle, position, and timing to comply with atmospheric refraction"; the formulas are in the paper's
 * ref. [7], not available, so this is the first-order planar-Snell reading): n(z) sin(theta(z)) is constant along the
 * ray, theta from the vertical.  To first order in eta = n - 1, for a ray leaving e_z at theta0 and reaching c_z < e_z:
 *   theta(z) - theta0 = tan(theta0) (eta(e_z) - eta(z))
 *   horizontal displacement beyond the straight line,
 *   dr = int (tan theta(z) - tan theta0) dz = tan(theta0) / cos^2(theta0) * [ eta(e_z) (e_z - c_z) - int_{c_z}^{e_z} eta dz ],
 *   int eta dz = 0.01 (eta0 / rho0) (T(c_z) - T(e_z))  [m]   (the same column integral as the delay of R8)
 *   dtheta = tan(theta0) (eta(e_z) - eta(c_z)).
 * Both are negative going down (the air gets denser: the ray bends towards the vertical).  The optical path changes
 * only to second order (Fermat), so the arrival time of R8 stands. */
#define ORC_REFRACT_VZ_MIN 0.25   /* cos(75.5 deg): where the first-order forms leave their 3e-3 bound (see below) */

void orc_refraction(const orc_atmosphere *atm, double e_z, double c_z, double v_z, double *dr, double *dtheta)
{
    double cos0 = fabs(v_z), sin0 = sqrt(fmax(0.0, 1.0 - v_z * v_z)), tan0 = sin0 / cos0;
    double eta_e = orc_refractivity(atm, e_z), eta_c = orc_refractivity(atm, c_z);
    double col = 0.01 * (atm->eta0 / atm->rho0) * (orc_depth(atm, c_z) - orc_depth(atm, e_z));
    *dr = tan0 / (cos0 * cos0) * (eta_e * (e_z - c_z) - col);
    *dtheta = tan0 * (eta_e - eta_c);
}

/* R10 / R11 with the corrections of R27 applied on the plane z = c_z: the arrival point moves by dr along the
 * horizontal direction of flight, the direction turns by dtheta in the vertical plane of flight; the sphere test
 * uses the corrected point and direction (q = corrected plane point - centre, q_z = 0):
 *   b^2 = |q|^2 - (q . v')^2,  closest approach at s_pl - q . v' along the path. */
int orc_intersect_refracted(const orc_atmosphere *atm, const double e[3], const double v[3], const double tel[4],
                            double *b2, double *s_c, double *s_pl, double xy[2], double vout[3])
{
    vout[0] = v[0]; vout[1] = v[1]; vout[2] = v[2];
    *b2 = 0.0; *s_c = 0.0; *s_pl = 0.0; xy[0] = xy[1] = 0.0;
    if (!(v[2] < 0.0) || !(e[2] > tel[2])) return 0;
    double sp = (tel[2] - e[2]) / v[2];
    double x = e[0] + sp * v[0] - tel[0], y = e[1] + sp * v[1] - tel[1];
    double sin0 = sqrt(v[0] * v[0] + v[1] * v[1]);
    /* Validity of the first-order forms (R27): the terms they drop are O(eta tan^2 theta0) of the correction.  Against
     * a Snell ray integrated through the same n(z) they stay within 3e-3 of it up to a zenith angle of 75.5 degrees
     * (|v_z| >= 0.25) for emission altitudes up to 30 km, and leave that bound beyond (6e-3 at 80, 2e-2 at 85 degrees;
     * tests/test_oracle_pins.py::test_refraction_first_order_validity_bound).  Flatter rays keep the straight line. */
    if (sin0 > 0.0 && v[2] <= -ORC_REFRACT_VZ_MIN) {
        double dr, dth;
        orc_refraction(atm, e[2], tel[2], v[2], &dr, &dth);
        double hx = v[0] / sin0, hy = v[1] / sin0;
        double th = atan2(sin0, -v[2]) + dth;
        x += dr * hx; y += dr * hy;
        vout[0] = sin(th) * hx; vout[1] = sin(th) * hy; vout[2] = -cos(th);
    }
    double qv = x * vout[0] + y * vout[1];
    *b2 = x * x + y * y - qv * qv;
    *s_c = sp - qv;
    *s_pl = sp;
    xy[0] = x; xy[1] = y;
    return (*b2 <= tel[3] * tel[3]) && (*s_c > 0.0);
}

/* R17: tau(h, lambda) bilinear in the table, clamped at the edges; survival
 * exp(-tau / |v_z|) applied as a weight factor. */
double orc_optical_depth(const orc_atmosphere *atm, double h, double lam)
{
    if (atm->tau_nh <= 0 || atm->tau == NULL) return 0.0;
    int nh = atm->tau_nh, nl = atm->tau_nl;
    double fh = (h - atm->tau_h0) / atm->tau_dh, fl = (lam - atm->tau_l0) / atm->tau_dl;
    if (fh < 0.0) fh = 0.0; if (fh > (double)(nh - 1)) fh = (double)(nh - 1);
    if (fl < 0.0) fl = 0.0; if (fl > (double)(nl - 1)) fl = (double)(nl - 1);
    int ih = (int)floor(fh), il = (int)floor(fl);
    if (ih > nh - 2) ih = nh - 2; if (ih < 0) ih = 0;
    if (il > nl - 2) il = nl - 2; if (il < 0) il = 0;
    double th = fh - ih, tl = fl - il;
    int ih1 = (nh > 1) ? ih + 1 : ih, il1 = (nl > 1) ? il + 1 : il;
    double t00 = atm->tau[ih * nl + il], t01 = atm->tau[ih * nl + il1];
    double t10 = atm->tau[ih1 * nl + il], t11 = atm->tau[ih1 * nl + il1];
    return (1.0 - th) * ((1.0 - tl) * t00 + tl * t01) + th * ((1.0 - tl) * t10 + tl * t11);
}

double orc_transmission(const orc_atmosphere *atm, double h, double lam, double v_z)
{
    return exp(-orc_optical_depth(atm, h, lam) / fabs(v_z));
}

/* ---------------------------------------------------------------------- */
/* The whole path over segments [0, n) with global ids first_id + i
 * (SURVEY.md §8(c) "Algorithm (oracle order of operations)").
 *
 *   counts   : NULL or uint32[n][2]  (n_b for tag 0 and tag 1)
 *   tallies  : orc_tally[n_tel], accumulated into
 *   counters : uint64[8] accumulated into:
 *              0 segments, 1 photons generated, 2 upward (v_z >= 0), 3 hits,
 *              4 records stored, 5 records dropped (capacity), 6 invalid segments, 7 bunches of cut segments (R29)
 *   records  : NULL or orc_record[cap]; *n_rec is advanced
 * Brute force over ALL telescopes; a photon may hit several; no shadowing (R10).
 */
/* R28: the sphere that holds every telescope sphere: centre = centre of the bounding box of the telescope centres,
 * R_b = max_k (|c_k - centre| + R_k). */
void orc_array_sphere(const double *tel, int n_tel, double out[4])
{
    double lo[3] = { INFINITY, INFINITY, INFINITY }, hi[3] = { -INFINITY, -INFINITY, -INFINITY };
    for (int k = 0; k < n_tel; ++k)
        for (int i = 0; i < 3; ++i) { lo[i] = fmin(lo[i], tel[4 * k + i]); hi[i] = fmax(hi[i], tel[4 * k + i]); }
    for (int i = 0; i < 3; ++i) out[i] = 0.5 * (lo[i] + hi[i]);
    double rb = 0.0;
    for (int k = 0; k < n_tel; ++k) {
        double x = tel[4 * k] - out[0], y = tel[4 * k + 1] - out[1], z = tel[4 * k + 2] - out[2];
        rb = fmax(rb, sqrt(x * x + y * y + z * z) + tel[4 * k + 3]);
    }
    out[3] = rb;
}

/* R29, the angular particle cut of PAPER.md:57 (section 1.2.1, Fig. 2): "calculate the angle difference between the
 * currently handled particles' flight direction and the vector to the experiment center.  For higher precision, the
 * minimum angle to each individual telescope can be used."  A Cherenkov segment is not handled (no photon is drawn)
 * when that angle exceeds the cut.  The vector is taken from the segment midpoint m = p0 + (L/2) d; the experiment
 * centre is the centre of the bounding box of the telescope centres (the point of R28).  angle(d, u) > cut is decided
 * as d.u < cos(cut) |u|, so that no inverse cosine enters.  Returns 1 when the segment is cut.  The cut is lossy: it
 * is the paper's trade of photons for speed, unlike the exact culling of the GPU path, which the oracle never needs. */
int orc_particle_cut(const double p0[3], const double d[3], double L, const double *tel, int n_tel, const double centre[3],
                     int mode, double cut_angle)
{
    if (mode == 0) return 0;
    double cc = cos(cut_angle);
    int n = (mode == 2) ? n_tel : 1;
    for (int k = 0; k < n; ++k) {
        const double *c = (mode == 2) ? &tel[4 * k] : centre;
        double u[3];
        for (int i = 0; i < 3; ++i) u[i] = c[i] - (p0[i] + (0.5 * L) * d[i]);
        double dot = (d[0] * u[0] + d[1] * u[1]) + d[2] * u[2];
        double norm = sqrt((u[0] * u[0] + u[1] * u[1]) + u[2] * u[2]);
        if (!(dot < cc * norm)) return 0;          /* within the cut of this target: the segment is handled */
    }
    return 1;
}

void orc_run(const orc_atmosphere *atm, const double *tel, int n_tel,
             const orc_segment *seg, uint64_t n, uint64_t first_id, const orc_params *par,
             uint32_t *counts, orc_tally *tallies, uint64_t *counters,
             orc_record *records, uint64_t cap, uint64_t *n_rec)
{
    double array[4];
    orc_array_sphere(tel, n_tel, array);
    for (uint64_t i = 0; i < n; ++i) {
        uint64_t S = first_id + i;
        counters[0] += 1;
        int invalid = 0;
        for (int tag = 0; tag < 2; ++tag) {
            if (counts) counts[2 * i + tag] = 0;
            if (!((par->processes >> tag) & 1u)) continue;
            orc_frame f;
            const double *bt = (tag == 1 && par->fl_beam_telescope >= 0) ? &tel[4 * par->fl_beam_telescope]
                             : (tag == 1 && par->fl_beam_telescope == -2) ? array : NULL;
            if (orc_preamble(atm, par, &seg[i], tag, bt, &f) != 0) { invalid = 1; continue; }
            if (counts) counts[2 * i + tag] = f.n_b;
            if (tag == 0 && orc_particle_cut(f.p0, f.d, f.L, tel, n_tel, array, par->cut_mode, par->cut_angle)) {
                counters[1] += f.n_b;          /* the bunches of a cut segment count as generated ... */
                counters[7] += f.n_b;          /* ... and as skipped */
                continue;
            }
            for (uint32_t j = 0; j < f.n_b; ++j) {
                orc_photon ph;
                orc_make_photon(&f, par, S, j, tag, &ph);
                counters[1] += 1;
                if (par->cauchy_b > 0.0 && tag == 0 && !(ph.w > 0.0)) continue;   /* R30: below the threshold at its wavelength */
                if (!(ph.v[2] < 0.0)) { counters[2] += 1; continue; }
                for (int k = 0; k < n_tel; ++k) {
                    double b2, s_c, s_pl, xy[2], va[3] = { ph.v[0], ph.v[1], ph.v[2] };
                    if (par->refract) {
                        if (!orc_intersect_refracted(atm, ph.e, ph.v, &tel[4 * k], &b2, &s_c, &s_pl, xy, va)) continue;
                    } else if (!orc_intersect(ph.e, ph.v, &tel[4 * k], &b2, &s_c, &s_pl, xy)) continue;
                    double t = orc_arrival_time(atm, ph.e[2], tel[4 * k + 2], ph.v[2], s_pl, ph.t_e);
                    double w = ph.w * orc_transmission(atm, ph.e[2], ph.lam, ph.v[2]);
                    tallies[k].hits += 1;
                    tallies[k].sum_w += w;
                    tallies[k].sum_wt += w * t;
                    counters[3] += 1;
                    if (records) {
                        if (*n_rec < cap) {
                            orc_record *r = &records[*n_rec];
                            r->x = xy[0]; r->y = xy[1]; r->cx = va[0]; r->cy = va[1];
                            r->t = t; r->lam = ph.lam; r->w = w;
                            r->id = (S << 25) | ((uint64_t)tag << 24) | (uint64_t)j;
                            r->tel = k; r->pad = 0;
                            *n_rec += 1;
                            counters[4] += 1;
                        } else {
                            counters[5] += 1;
                        }
                    }
                }
            }
        }
        if (invalid) counters[6] += 1;
    }
}
