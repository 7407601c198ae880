/*
 * sas_oracle.h -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, single-threaded fp64 CPU restatement of the SANS Monte-Carlo
 * hot path of arXiv 2501.06054, written from the paper and the
 * readings listed in DESIGN.md section 3.  It shares no code, header, table
 * or constant generator with the CUDA library under paper_2501_06054_b200/.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call it.
 *
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared  (no FMA contraction: every
 * written operation is individually rounded, DESIGN.md R-C0).
 *
 * Units: instrument geometry in metres, wavelengths in Angstrom, Q in 1/A,
 * particle sizes in A, contrasts in 1/A^2, intensity in 1/cm.
 */
#ifndef SAS_ORACLE_H
#define SAS_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* outcome of one neutron (PAPER.md:143-147 trace loop; DESIGN.md R-C4..R-C9) */
enum {
  ORC_DETECTED = 0,
  ORC_SLIT1 = 1,
  ORC_SLIT2 = 2,
  ORC_MISS_SAMPLE = 3,
  ORC_UNREACHABLE = 4,
  ORC_MISS_DET = 5
};

enum { ORC_SAMPLE_BOX = 0, ORC_SAMPLE_CYL_Y = 1 };
/* R-L1: uniform band (BASELINE.json configs), or the triangular transmission of a mechanical velocity selector
 * (KWS-1's selector sets the wavelength spread): symmetric triangle on [lambda_min, lambda_max] */
enum { ORC_LAMBDA_UNIFORM = 0, ORC_LAMBDA_TRIANGLE = 1 };
enum {
  ORC_SPHERE = 0,
  ORC_CORE_SHELL_SPHERE = 1,
  ORC_CYLINDER = 2,
  ORC_TRIAXIAL = 3,
  ORC_CORE_SHELL_TRIAXIAL = 4,
  ORC_FLAT = 5,
  /* NEXT-2: three more of the paper's models, each Eq. 1 integrated over its body */
  ORC_PARALLELEPIPED = 6,       /* Table I group E, Eq. 6: sides a, b, c along A, B, C */
  ORC_CORE_SHELL_CYLINDER = 7,  /* Table I group A, Eq. 7: core R, L; shell t on every face */
  ORC_ELLIPSOID = 8,            /* Table I group B, Eq. 7: equatorial R_e, polar R_p (axis C) */
  /* two of the models the paper found expensive (inner numerical integration; R-M2):
   * bodies of revolution = cylinder (R, L) + two spherical end pieces of radius R_b >= R, Eq. 1 integrated
   * slice by slice with a 32-node Gauss-Legendre rule over each end piece */
  ORC_BARBELL = 9,              /* sphere centres outside the cylinder, at +-(L/2 + h), h = sqrt(R_b^2 - R^2) */
  ORC_CAPPED_CYLINDER = 10,     /* sphere centres inside, at +-(L/2 - h): lens-shaped caps */
  /* three more bodies of Table I, each Eq. 1 over the body (R-M3) */
  ORC_ELLIPTICAL_CYLINDER = 11, /* group B: cross-section semi-axes a (along A), b (along B), length L along C */
  ORC_HOLLOW_CYLINDER = 12,     /* group A: tube, hollow core radius R, wall thickness t, length L */
  ORC_CORE_SHELL_ELLIPSOID = 13, /* group B: core of revolution (R_e, R_p) in a shell of thickness t */
  /* one of the models the paper found expensive (Table II group F "Polymer micelle"): a homogeneous
   * spherical core with N Gaussian chains attached to its surface (Pedersen & Gerstenberg, Macromolecules 29
   * (1996) 1363; DESIGN.md R-M4).  size = R_core, R_g, V_chain (A^3), N; sld[0] core, sld[1] chain */
  ORC_POLYMER_MICELLE = 14,
  /* another of them ("Hollow rectangular prism thin walls"; DESIGN.md R-M5): a rectangular prism
   * a x b x c whose contrast sits in infinitely thin walls on its six faces: Eq. 1 as a surface integral, to first
   * order in the wall thickness t.  size = a, b, c, t; sld[0] wall contrast; pd[0] = common scale of a, b, c */
  ORC_HOLLOW_PRISM_THIN = 15
};
enum {
  ORC_ORIENT_FIXED = 0,
  ORC_ORIENT_GAUSS_QUAD = 1,
  ORC_ORIENT_ISOTROPIC_MC = 2,
  ORC_ORIENT_UNIFORM_ANGLES_MC = 3 /* PAPER.md:131-133 as printed: theta~U[0,pi], phi, psi~U[0,2pi] (R-N3) */
};
/* ORC_SQ_HAYTER_MSA (R-S2; Table II group F "Hayter MSA"): mean-spherical closure for hard spheres of
 * diameter 2 sq_radius_eff with a screened-Coulomb (Yukawa) repulsion of contact value sq_contact_kT and inverse
 * screening length sq_kappa_sigma (in units of the diameter) */
enum { ORC_SQ_NONE = 0, ORC_SQ_HARD_SPHERE_PY = 1, ORC_SQ_HAYTER_MSA = 2 };

#define ORC_MAX_NODES 64

/* Instrument: PAPER.md:86 (source, slits, sample, 2-D PSD). */
typedef struct {
  double src_xw, src_yh;          /* flat source, m */
  double lambda_min, lambda_max;  /* A */
  double flux;
  double slit1_z, slit1_xw, slit1_yh;
  double slit2_z, slit2_xw, slit2_yh;
  double focus_z, focus_xw, focus_yh;
  int32_t sample_shape;
  int32_t lambda_dist;            /* ORC_LAMBDA_*: law of the wavelength inside [lambda_min, lambda_max] (R-L1) */
  double sample_z, sample_xw, sample_yh, sample_zd, sample_radius;
  double mu_abs_2200, mu_inc;     /* 1/m */
  double q_min, q_max;            /* 1/A */
  double det_dist, det_xw, det_yh;
  int32_t det_nx, det_ny;
} orc_instrument;

/* Sample model with its quadrature tables already expanded by the caller
 * (oracle/oracle.py builds them with numpy: DESIGN.md R-A9, R-A11). */
typedef struct {
  int32_t model;
  int32_t orient_kind;
  int32_t sq_kind;
  int32_t pad0;
  double scale, background;
  double sld[3];
  double size[4];
  /* polydispersity: two tensor axes of relative-size nodes (value, weight);
   * n_pd[k]=1 with node 1.0 / weight 1.0 means monodisperse. The node value
   * multiplies size[...] as DESIGN.md R-A12 states per model. */
  int32_t n_pd[2];
  double pd_x[2][ORC_MAX_NODES];
  double pd_w[2][ORC_MAX_NODES];
  /* orientation */
  double theta, phi, psi;         /* rad */
  int32_t n_or[2];                /* Gauss quadrature tilts (theta, phi) */
  double or_d[2][ORC_MAX_NODES];  /* tilt angle Delta (rad) */
  double or_w[2][ORC_MAX_NODES];
  double sq_radius_eff, sq_volfrac;
  /* The paper's own polydispersity (Eq. 8; DESIGN.md R-N1, R-N2): pd_mc[k] != 0 draws
   * length k of every scattering event from N(mean, (pd_rel[k] mean)^2), redrawn while not positive;
   * the fixed-node tables of axis k must then be the single node (1.0, 1.0). */
  int32_t pd_mc[2];
  double pd_rel[2];
  /* R-S2: the caller (oracle/oracle.py: msa_solve) solved the closure: Baxter function inside the core
   * Q(x) = a (x^2 - 1)/2 + b (x - 1) + E exp(-k x) - C', outside D' exp(-k (x - 1)); msa = {a, b, E, C', D'} */
  double sq_contact_kT, sq_kappa_sigma;
  double msa[5];
} orc_model;

/* full per-neutron record, for pins and parity */
typedef struct {
  int32_t status;
  int32_t pixel;       /* iy*nx+ix, or -1 */
  double weight;       /* p   (R-C11) */
  double weight_env;   /* p with every shape factor Phi, sinc, Lambda := 1 (R-C15) */
  double q;            /* sampled |Q| */
  double Q[3];
  double lambda;
  double ell;          /* chord length in the sample, m */
  double p0;           /* source weight */
  double intensity;    /* I(Q) 1/cm */
  double u[12];        /* the uniforms drawn (unused ones stay 0) */
  double pd_x[2];      /* relative sizes drawn for this event (1 when the axis is not sampled) */
  int32_t pd_tries[2]; /* Philox blocks used by each sampled axis (1 = no redraw) */
} orc_record;

/* Philox4x32-10, Salmon et al. SC'11 (DESIGN.md R-B). */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double orc_uniform(uint32_t word);

/* R-M4 pieces: Debye function of a Gaussian chain D(x) = 2 (exp(-x) - 1 + x) / x^2, its amplitude relative to a
 * chain end psi(x) = (1 - exp(-x)) / x, x = (q R_g)^2, and the micelle's |F|^2 (not a perfect square: the chains'
 * self term is the Debye function); *vol = V_core + N V_chain, *env2 = the same with every shape factor 1 */
double orc_debye(double x);
double orc_chain_psi(double x);
double orc_micelle_f2(const orc_model* m, double q, double x0, double* vol, double* env2);

/* R-S2: S(q) = 1 / |Qhat(K)|^2, K = 2 q R_eff, Qhat(K) = 1 - 12 eta int_0^inf Q(x) exp(i K x) dx: the core part by the
 * 64-node Gauss-Legendre rule, the tail in closed form */
double orc_msa_sq(double q, const orc_model* m);

/* form / structure factor pieces (PAPER.md:37-49 Eq.1-4, :161-163 Eq.9) */
double orc_sphere_phi(double u);                 /* 3(sin u - u cos u)/u^3 */
double orc_sinc(double x);
double orc_lambda1(double x);                    /* 2 J1(x)/x */
double orc_py_sq(double q, double r_eff, double volfrac);
/* I(Q) in 1/cm for a Q vector given in the GLOBAL frame, with orientation
 * uniforms u_or[3] (used only by ORC_ORIENT_ISOTROPIC_MC). env (nullable)
 * receives the envelope intensity. */
double orc_intensity(const orc_model* m, const double Q[3], const double u_or[3], double* env);
/* The per-event form of the paper (Eq. 4 with the event's own sizes, R-N2): relative sizes x[2] given. */
double orc_intensity_event(const orc_model* m, const double Q[3], const double u_or[3], const double x[2],
                           double* env);
/* Relative size of axis k of event (seed, id, exp) by R-N1; *tries = Philox blocks consumed. */
double orc_draw_rel_size(uint64_t seed, uint64_t id, uint32_t exp_index, int k, double rel, int32_t* tries);
/* amplitude F (A^-2 * A^3) of one particle with explicit axes projections */
double orc_amplitude(const orc_model* m, double qa, double qb, double qc, double x0, double x1,
                     double* vol, double* env);

/* one neutron */
void orc_trace_one(const orc_instrument* ins, const orc_model* m, uint64_t seed, uint64_t id,
                   uint32_t exp_index, orc_record* rec);

/* ids [first, first+n): optional per-neutron dumps (nullable), optional
 * histograms (nullable, accumulated in id order: R-C14), counters[8]
 * (launched, slit1, slit2, miss_sample, unreachable, miss_det, detected, 0)
 * are incremented. */
void orc_trace_range(const orc_instrument* ins, const orc_model* m, uint64_t seed, uint64_t first,
                     uint64_t n, uint32_t exp_index, int32_t* pixel, double* weight, double* weight_env,
                     double* q, double* sum_p, double* sum_p2, uint64_t* counts, uint64_t counters[8]);

/* NEXT-4, reading R-R1 of DESIGN.md: ring average of one detector image into I(q) with its
 * standard error (PAPER.md:86 2-D PSD, :173 I(Q) curve against a measurement).  Pixel centre (X, Y) ->
 * two_theta = atan2(sqrt(X^2+Y^2), D), q = (2 k) sin(two_theta / 2), k = TWO_PI / lambda_ref; pixel solid angle
 * dOmega = A_pix D / (D^2+r^2)^(3/2); bin b = floor((q - q_lo) n_bins / (q_hi - q_lo)) for q_lo <= q < q_hi;
 * I_b = sum P / (sum dOmega * launched), sigma_b = sqrt(sum P2) / (sum dOmega * launched), q_b = bin centre,
 * npix_b = pixels in the ring (empty ring: I = sigma = 0). */
void orc_reduce_radial(const orc_instrument* ins, const double* sum_p, const double* sum_p2, double launched,
                       double lambda_ref, double q_lo, double q_hi, int32_t n_bins, double* q_out, double* i_out,
                       double* sigma_out, uint64_t* npix_out);

#ifdef __cplusplus
}
#endif
#endif
