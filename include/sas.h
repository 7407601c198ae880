/*
 * sas.h -- C ABI of the B200-native SANS Monte-Carlo tracer (libsas_b200.so).
 *
 * The library traces neutrons of a small-angle-scattering virtual experiment
 * (PAPER.md:19, :86, :143-147 -- arXiv 2501.06054): source -> two slits ->
 * sample -> choose Q -> weight by the SAS model intensity I(Q) (PAPER.md:37-49,
 * Eq. 1-4; :161-163, Eq. 9; polydispersity and orientation distributions
 * :122-135) -> 2-D position-sensitive detector histogram.  Every step runs in
 * hand-written CUDA kernels for sm_100a; there is no CPU fallback: a call that
 * cannot run on the device returns SAS_ECUDA.
 *
 * Conventions
 *   - Plain C, no exceptions cross the boundary; every call returns sas_status
 *     (SAS_OK == 0) and leaves a message readable with sas_last_error().
 *   - "h_" pointers are HOST memory, "d_" pointers are DEVICE memory of the
 *     current CUDA device, both caller-owned and caller-sized unless said
 *     otherwise.  Descriptors are host structs, copied by the call.
 *   - Instrument lengths are metres; wavelengths Angstrom; Q in 1/Angstrom;
 *     particle sizes Angstrom; contrasts 1/Angstrom^2; intensities 1/cm;
 *     angles radians.
 *   - Detector arrays are row-major [ny][nx], index = iy*nx + ix; in batched
 *     mode [n_exp][ny][nx].  sum_p and sum_p2 are double, counts uint64_t.
 *   - Weights carry no 1/N: the weight of a neutron depends only on
 *     (seed, id, experiment index) and the descriptors, so id ranges are
 *     additive; normalise with counters[0] (launched).
 *   - sas_trace* enqueue on the context's stream and return; sas_read_detector
 *     and sas_get_counters synchronise that stream.
 *   - A context is not thread-safe; distinct contexts are independent.
 *   - The precise arithmetic (draw table, operation order) is DESIGN.md s.3.
 */
#ifndef SAS_H
#define SAS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sas_ctx sas_ctx; /* opaque; owns device constants, tables, counters */

typedef enum {
  SAS_OK = 0,
  SAS_EINVAL = 1,       /* bad descriptor or argument */
  SAS_ESTATE = 2,       /* call out of order (e.g. trace before set_model) */
  SAS_ECUDA = 3,        /* CUDA runtime failure, or no usable device */
  SAS_ENOMEM = 4,
  SAS_EUNSUPPORTED = 5  /* valid request this build does not implement */
} sas_status;

/* precision of the MODEL evaluation; RNG->uniform and geometry are always fp64.  SAS_FP32 is a request: an
 * experiment whose model is evaluated once per neutron (no node loop), or whose phases q_max x size exceed 1e3
 * rad (the proven range of the fp32 argument reductions), runs its model in fp64. */
enum { SAS_FP32 = 0, SAS_FP64 = 1 };
enum { SAS_SAMPLE_BOX = 0, SAS_SAMPLE_CYL_Y = 1 };
/* law of the wavelength inside [lambda_min, lambda_max] (DESIGN.md R-L1): uniform, or the symmetric triangle of a
 * mechanical velocity selector, FWHM = (lambda_max - lambda_min) / 2 */
enum { SAS_LAMBDA_UNIFORM = 0, SAS_LAMBDA_TRIANGLE = 1 };
enum {
  SAS_SPHERE = 0,              /* Table II F.9 */
  SAS_CORE_SHELL_SPHERE = 1,   /* Table II F.3  */
  SAS_CYLINDER = 2,            /* Table I  A.7, Eq. 9 */
  SAS_TRIAXIAL_ELLIPSOID = 3,  /* Table I  B.3  */
  SAS_CORE_SHELL_TRIAXIAL = 4, /* B.3's shape with B.1's two-contrast composition (DESIGN.md R-A12) */
  SAS_FLAT = 5,                /* I == scale + background: test model */
  /* NEXT-2: evaluated in fp64 whatever `precision` says; orientation fixed or per event
   * (no SAS_ORIENT_GAUSS_QUAD) */
  SAS_PARALLELEPIPED = 6,      /* size = a, b, c along A, B, C (Eq. 6); pd[0] = common scale */
  SAS_CORE_SHELL_CYLINDER = 7, /* size = R, L, t (Eq. 7); sld[0] core, sld[1] shell; pd[0] on R, pd[1] on L */
  SAS_ELLIPSOID = 8,           /* size = R_equatorial, R_polar (axis C, Eq. 7); pd[0] on R_e, pd[1] on R_p */
  /* two of the models the paper found expensive (DESIGN.md R-M2): cylinder (R, L) along C plus two
   * spherical end pieces of radius R_b >= R, integrated slice by slice (32 Gauss-Legendre nodes per end piece).
   * size = R, L, R_b; pd[0] on R, pd[1] on L */
  SAS_BARBELL = 9,             /* sphere centres outside the cylinder, at +-(L/2 + sqrt(R_b^2 - R^2)) */
  SAS_CAPPED_CYLINDER = 10,    /* sphere centres inside, at +-(L/2 - sqrt(R_b^2 - R^2)): lens-shaped caps */
  /* three more bodies of Table I (DESIGN.md R-M3) */
  SAS_ELLIPTICAL_CYLINDER = 11,  /* size = a (along A), b (along B), L (along C); pd[0] scales a and b, pd[1] on L */
  SAS_HOLLOW_CYLINDER = 12,      /* size = hollow core radius R, L, wall thickness t; pd[0] on R, pd[1] on L */
  SAS_CORE_SHELL_ELLIPSOID = 13, /* size = R_e, R_p, t; sld[0] core, sld[1] shell; pd[0] on R_e, pd[1] on R_p */
  /* polymer micelle (PAPER.md:201 and Table II group F name it among the expensive models; DESIGN.md R-M4:
   * Pedersen & Gerstenberg, Macromolecules 29 (1996) 1363): homogeneous spherical core with N Gaussian chains
   * starting at R_core + R_g.  size = R_core, R_g, V_chain (A^3), N (0 or >= 1); sld[0] core, sld[1] chain
   * contrast; normalising volume V_core + N V_chain; pd[0] on R_core; isotropic (orientation is ignored) */
  SAS_POLYMER_MICELLE = 14,
  /* thin-walled hollow rectangular prism (PAPER.md:201 names it among the expensive models; DESIGN.md R-M5): a prism
   * a x b x c along A, B, C whose contrast sld[0] sits in walls of thickness t on its six faces, to first order in t
   * (Eq. 1 as a surface integral).  size = a, b, c, t; normalising volume = wall volume 2 t (ab + bc + ca);
   * pd[0] = common scale of a, b, c */
  SAS_HOLLOW_PRISM_THIN = 15
};
enum {
  SAS_ORIENT_FIXED = 0,
  SAS_ORIENT_GAUSS_QUAD = 1,
  SAS_ORIENT_ISOTROPIC_MC = 2,
  /* the paper's printed law, one draw per scattering event: theta ~ U[0,pi], phi, psi ~ U[0,2pi]
   * (DESIGN.md R-N3: not isotropic) */
  SAS_ORIENT_UNIFORM_ANGLES_MC = 3
};
enum {
  SAS_PD_NONE = 0,
  SAS_PD_SCHULZ_QUAD = 1,
  /* the paper's own averaging (Eq. 8; DESIGN.md R-N1, R-N2): one size per scattering
   * event from N(mean, (pd_rel mean)^2), redrawn while not positive; the event's intensity is Eq. 4 with
   * the event's own volume.  Does not combine with SAS_PD_SCHULZ_QUAD or SAS_ORIENT_GAUSS_QUAD
   * (SAS_EUNSUPPORTED); evaluated in fp64 whatever `precision` says. */
  SAS_PD_GAUSS_MC = 2
};
enum {
  SAS_SQ_NONE = 0,
  SAS_SQ_HARD_SPHERE_PY = 1,
  /* Hayter-Penfold MSA (Table II group F; DESIGN.md R-S2): mean-spherical closure for hard spheres of
   * radius sq_radius_eff and packing sq_volfrac with a screened-Coulomb repulsion of contact value sq_contact_kT
   * (in kT) and inverse screening length sq_kappa_sigma (in units of 1/diameter), solved on the host through the
   * Baxter / Hoye-Blum factorisation; S(q) by a 64-node Gauss-Legendre rule on the device, once per detected
   * neutron.  Offered for the globular models (sphere, core-shell sphere, the ellipsoids, polymer micelle); the
   * rod- and plate-like models refuse it.  SAS_EUNSUPPORTED: such a model, 2 q_max sq_radius_eff > 64 (beyond the rule's range), a contact value g(1+) < 0
   * (the closure's known failure for dilute, strongly charged systems; the rescaled MSA is not implemented), or no
   * convergence. */
  SAS_SQ_HAYTER_MSA = 2
};

#define SAS_MAX_NODES 64      /* per quadrature axis */
#define SAS_MAX_PD_PAIRS 1024 /* pd_nodes[0]*pd_nodes[1] */

/* Instrument (source, slits defining the divergence, sample, 2-D PSD). */
typedef struct {
  uint32_t struct_size;              /* = sizeof(sas_instrument_desc) */
  int32_t sample_shape;              /* SAS_SAMPLE_* */
  double src_xw, src_yh;             /* flat rectangular source in the plane z = 0 */
  double lambda_min, lambda_max;     /* wavelength band (law: lambda_dist); equal => monochromatic */
  double flux;                       /* n / (cm^2 s sr A); 1 for unit flux */
  double slit1_z, slit1_xw, slit1_yh;
  double slit2_z, slit2_xw, slit2_yh;
  double focus_z, focus_xw, focus_yh; /* rectangle the source aims at, uniformly (normally slit 2) */
  double sample_z;                   /* sample centre */
  double sample_xw, sample_yh, sample_zd; /* box extents; yh is also the cylinder height */
  double sample_radius;              /* SAS_SAMPLE_CYL_Y: axis along y */
  double mu_abs_2200, mu_inc;        /* 1/m; absorption at 1.7982 A (scaled ~lambda) and incoherent; 0 => no attenuation */
  double q_min, q_max;               /* |Q| is drawn uniformly in [q_min, q_max] */
  double det_dist;                   /* detector plane at sample_z + det_dist */
  double det_xw, det_yh;
  int32_t det_nx, det_ny;
  int32_t lambda_dist;               /* SAS_LAMBDA_* */
  int32_t reserved;
} sas_instrument_desc;

/* Sample model (PAPER.md:51 parameters {theta_i}; :122-133 distributions). */
typedef struct {
  uint32_t struct_size;              /* = sizeof(sas_model_desc) */
  int32_t model;                     /* SAS_SPHERE ... */
  int32_t precision;                 /* SAS_FP32 | SAS_FP64 */
  int32_t orient_kind;               /* SAS_ORIENT_* */
  int32_t sq_kind;                   /* SAS_SQ_* */
  int32_t pd_kind[2];                /* SAS_PD_* for the two polydisperse lengths */
  int32_t pd_nodes[2];               /* quadrature nodes (1..SAS_MAX_NODES) */
  int32_t n_theta, n_phi;            /* SAS_ORIENT_GAUSS_QUAD nodes */
  int32_t reserved;
  double scale, background;          /* scale = volume fraction; background 1/cm */
  double sld[3];                     /* contrast vs solvent: [0] particle/core, [1] shell */
  double size[4];                    /* sphere R | core-shell Rc,t | cylinder R,L | a,b,c | a,b,c,t */
  double pd_rel[2];                  /* sigma/mean of: [0] R|Rc|R|common scale of (a,b,c); [1] t|L|t */
  double theta, phi, psi;            /* axis polar angle from +z, azimuth from +x, spin (DESIGN.md R-A7) */
  double sigma_theta, sigma_phi;     /* Gaussian spreads of the two tilts (uniaxial models only) */
  double sq_radius_eff, sq_volfrac;  /* Percus-Yevick hard-sphere S(q) (Table II F.11) */
  double sq_contact_kT, sq_kappa_sigma; /* SAS_SQ_HAYTER_MSA only: beta u at contact, kappa x diameter */
} sas_model_desc;

/* --- single experiment --------------------------------------------------- */

/* Validate and copy the instrument; allocate device state on the current CUDA
 * device (its own zeroed histograms and an internal stream until sas_bind_buffers
 * says otherwise).  *out is set only on SAS_OK; free with sas_destroy.  The context stays on that device:
 * every later call on it runs there whatever the calling thread's current device is (and leaves that unchanged). */
sas_status sas_create_instrument(const sas_instrument_desc* instr, sas_ctx** out);

/* Use caller-owned DEVICE histograms ([n_exp][ny][nx]: double, double, uint64)
 * and CUDA stream (a cudaStream_t passed as void*; NULL = default stream).
 * The caller keeps ownership and must keep them alive; contents are not cleared. */
sas_status sas_bind_buffers(sas_ctx* ctx, void* d_sum_p, void* d_sum_p2, void* d_counts, void* cuda_stream);

/* Validate the model, build the quadrature tables on the host (generalised
 * Gauss-Laguerre for Schulz sizes, Gauss-Legendre for Gaussian tilts;
 * DESIGN.md R-A9, R-A11) and upload them (asynchronous H2D on the stream). */
sas_status sas_set_model(sas_ctx* ctx, const sas_model_desc* model);

/* Trace neutron ids [0, n) (sas_trace) or [first_id, first_id+n) and ACCUMULATE
 * into the histograms and counters (PAPER.md:143-147 trace loop). */
sas_status sas_trace(sas_ctx* ctx, uint64_t n_neutrons, uint64_t seed);
sas_status sas_trace_range(sas_ctx* ctx, uint64_t first_id, uint64_t n, uint64_t seed);

/* Parity hook: no histogram; writes, for id = first_id + i, d_pixel[i] (iy*nx+ix,
 * or -1 when the neutron is not detected), d_weight[i] (0 when not detected) and,
 * if d_q is not NULL, the drawn |Q| (0 if the neutron died before the draw).
 * Single-experiment contexts only; exp_index enters the Philox counter. n <= 2^31. */
sas_status sas_trace_dump(sas_ctx* ctx, uint64_t first_id, uint64_t n, uint64_t seed, uint32_t exp_index,
                          int32_t* d_pixel, double* d_weight, double* d_q);

/* Synchronise and copy the histograms to HOST arrays (any may be NULL). */
sas_status sas_read_detector(sas_ctx* ctx, double* h_sum_p, double* h_sum_p2, uint64_t* h_counts);

/* out[8] = launched, absorbed at slit 1, at slit 2, missed the sample, |Q| unreachable
 * (q >= 2k), missed the detector, detected; out[7] = how many of the detector misses (out[5])
 * were decided by the conservative q*lambda classifier without running the full geometry
 * (an implementation statistic).  Summed over experiments.  Synchronises.
 * out[0] is the library's own sum of the traced ranges; the kernels count every outcome they decide in
 * their queued stages and out[1] is what is left of out[0] (a neutron has exactly one outcome), so
 * out[0] == out[1] + ... + out[6] always. */
sas_status sas_get_counters(sas_ctx* ctx, uint64_t out[8]);

/* Zero histograms and counters (asynchronous on the stream). */
sas_status sas_reset_detector(sas_ctx* ctx);

void sas_destroy(sas_ctx* ctx);
/* Message of the last failing call on ctx (or of the last failing create when ctx == NULL). */
const char* sas_last_error(const sas_ctx* ctx);

/* --- batched mode (PAPER.md:19, :213 dataset generation) ------------------ */

/* n_exp experiments, each with its own instrument + model and its own histogram
 * ([n_exp][ny][nx]; every experiment must have the same det_nx, det_ny).  Tables are built and
 * uploaded here.  Experiments are grouped by kernel (model form, per-event or fixed-node sizes, precision of the
 * model arithmetic): a trace call launches one kernel per group present. */
sas_status sas_create_batch(const sas_instrument_desc* instr, const sas_model_desc* model, uint32_t n_exp,
                            sas_ctx** out);
/* Trace ids [0, n_neutrons_each) of every experiment in ONE launch; experiment e
 * uses Philox counter word 3 = e. */
sas_status sas_trace_batch(sas_ctx* ctx, uint64_t n_neutrons_each, uint64_t seed);
/* The same for ids [first_id, first_id + n_each) of every experiment (accumulates): a batch can be resumed, or
 * sharded over GPUs by contiguous id ranges exactly like a single experiment (scatter
 * ncount/N, gather) -- the union of the ranges is the same set of neutrons as one call over the whole range. */
sas_status sas_trace_batch_range(sas_ctx* ctx, uint64_t first_id, uint64_t n_each, uint64_t seed);

/* --- introspection -------------------------------------------------------- */
/* HOST-ONLY (needs no device): the quadrature rule the library builds for
 * kind 0 = Schulz sizes of relative width param (values = size multipliers of mean 1;
 *          generalised Gauss-Laguerre, DESIGN.md R-A9),
 * kind 1 = Gaussian tilt of standard deviation param radians on [-3 sigma, 3 sigma]
 *          (values = tilt angles; Gauss-Legendre x Gaussian, DESIGN.md R-A11).
 * Writes n values and n weights (weights sum to 1).  n in 1..SAS_MAX_NODES. */
sas_status sas_quadrature_nodes(int32_t kind, double param, int32_t n, double* h_values, double* h_weights);
/* Number of kernel launches this context has issued, and launch geometry of the last one. */
sas_status sas_get_launch_info(sas_ctx* ctx, uint64_t* n_launches, int32_t* grid, int32_t* block,
                               int32_t* smem_bytes);
/* Average device time in ms (CUDA events on the context's stream) of the trace kernels launched
 * since the last call with reset != 0; *n_timed = how many launches the average covers. */
sas_status sas_get_kernel_time(sas_ctx* ctx, int32_t reset, double* avg_ms, uint64_t* n_timed);
/* Per-launch timing on (enabled != 0, the default) or off.  On, every trace-kernel launch is bracketed by two
 * cudaEventRecord on the context's stream -- about 6 us of stream operations per launch on a B200, which is a
 * quarter of a 1e6-neutron step (BASELINE.json configs[0]; PAPER.md:195 is about exactly such fixed costs).  Off,
 * a launch is the kernel alone: sas_get_kernel_time and sas_get_launch_records then report no launches.
 * Takes effect from the next launch; results are the same either way. */
sas_status sas_set_launch_timing(sas_ctx* ctx, int32_t enabled);
/* One record per trace-kernel launch since the last sas_get_kernel_time(reset != 0), oldest first (at most
 * SAS_MAX_LAUNCH_RECORDS are kept): which kernel ran (variant = the model form it was compiled for, per-event
 * sizes or fixed nodes, precision of the model arithmetic), over how many experiments and ids, and its device
 * time from CUDA events on the context's stream.  Writes min(*n, cap) records to h_records; synchronises. */
#define SAS_MAX_LAUNCH_RECORDS 4096
typedef struct {
  int32_t variant;       /* internal kernel variant: 0 sphere, 1 core-shell sphere, 2 cylinder, 3 triaxial,
                            4 core-shell triaxial, 5 flat, 6 cylinder with tilt quadrature, 7.. NEXT-2 models */
  int32_t per_event;     /* 1: SAS_PD_GAUSS_MC kernel */
  int32_t precision;     /* SAS_FP32 | SAS_FP64 actually used by the model arithmetic */
  int32_t warp_specialised; /* 1: producer/consumer kernel (trace_kernel_ws.cuh) */
  uint32_t n_exp;        /* experiments of the launch */
  uint32_t n_per_exp;    /* ids per experiment */
  int32_t grid, block;   /* block: 256 = one producer + one consumer warpgroup, 512 = one + three (launches bound by
                            the model evaluation; warp-specialised kernel), 128 = unified kernel */
  double ms;
} sas_launch_record;
sas_status sas_get_launch_records(sas_ctx* ctx, sas_launch_record* h_records, uint32_t cap, uint32_t* n);
/* Bytes of the last host-to-device upload of parameters and quadrature tables (sas_set_model /
 * sas_create_batch). */
sas_status sas_get_upload_bytes(sas_ctx* ctx, uint64_t* bytes);

/* ---- NEXT-4: data reduction of the virtual experiment ----
 * Ring average of the detector image of experiment `exp_index` into I(q) with its standard error
 * (PAPER.md:86 2-D PSD, :173 I(Q) curve; DESIGN.md R-R1).  Pixel centre (X, Y): two_theta = atan2(r, D),
 * q = (4 pi / lambda_ref) sin(two_theta / 2), solid angle dOmega = A_pix D / (D^2 + r^2)^(3/2); ring
 * b = floor((q - q_lo) n_bins / (q_hi - q_lo)) for q_lo <= q < q_hi.  Host outputs, n_bins entries each (any may
 * be NULL): q = ring centres, I = sum P / (sum dOmega * launched) (weight per steradian per launched neutron of
 * that experiment; launched = desc->n_launched, or the context's own count when that is 0), sigma = sqrt(sum P2) / (same), npix = pixels in the ring (empty ring: I = sigma = 0).
 * Runs one CUDA kernel on the context's stream over the bound histograms and synchronises.
 * SAS_EINVAL: n_bins outside 1..SAS_MAX_RINGS, q_lo >= q_hi, lambda_ref <= 0, exp_index out of range. */
#define SAS_MAX_RINGS 1024
typedef struct {
  uint32_t struct_size;
  uint32_t exp_index;
  int32_t n_bins;
  int32_t reserved;
  double q_lo, q_hi;      /* 1/A */
  double lambda_ref;      /* A: the wavelength that converts angle to q */
  uint64_t n_launched;    /* neutrons launched INTO THIS EXPERIMENT that the bound histograms hold; 0 = what this
                             context traced since its last reset / bind.  Must be given when the buffers hold more
                             than that (detectors merged from other GPUs, buffers accumulated elsewhere). */
} sas_radial_desc;
sas_status sas_reduce_radial(sas_ctx* ctx, const sas_radial_desc* desc, double* h_q, double* h_I, double* h_sigma,
                             uint64_t* h_npix);

/* The same ring average for callers that must not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): no context, no cudaMalloc / cudaFree / event creation / synchronisation -- one
 * cudaMemsetAsync and two kernel launches on `stream` (a cudaStream_t; NULL = the default stream) of the CURRENT
 * device.  The ring scratch is a static device array of SAS_STATIC_MAX_RINGS rings (16 KB) that every GPU which
 * loads the library holds until exit.
 *   ins       detector geometry (det_nx, det_ny, det_xw, det_yh, det_dist are read; struct_size checked)
 *   desc      as for sas_reduce_radial; exp_index is ignored; n_launched MUST be given (> 0)
 *   d_sum_p, d_sum_p2   DEVICE, [det_ny][det_nx] doubles of one experiment (inputs, caller-owned, not modified)
 *   d_q, d_I, d_sigma, d_npix   DEVICE outputs, n_bins entries each, caller-owned; any may be NULL
 * Asynchronous: outputs are valid once the work queued on `stream` has completed.  Results equal
 * sas_reduce_radial's (ring sums in a different order of fp64 additions: 1e-12; q and npix exactly).
 * All calls on a device share the static array, which keeps the last call's sums: every call first clears what it
 * uses, in stream order, so calls queued on ONE stream are safe back to back; calls that overlap on the GPU
 * (different streams without a dependency, or different host threads) RACE -- serialise them.  The first call on a
 * device looks the array's address up (once per device; make that call outside a graph capture).
 * SAS_EINVAL: n_bins outside 1..SAS_STATIC_MAX_RINGS (message names the limit; use sas_reduce_radial beyond it),
 * n_launched == 0, NULL inputs, bad geometry or q range; SAS_ECUDA: a CUDA call failed.  Message: sas_last_error(NULL). */
#define SAS_STATIC_MAX_RINGS 512
sas_status sas_reduce_radial_static(const sas_instrument_desc* ins, const sas_radial_desc* desc, const double* d_sum_p,
                                    const double* d_sum_p2, double* d_q, double* d_I, double* d_sigma,
                                    uint64_t* d_npix, void* stream);

/* Device time in ms (CUDA events around the kernel) of the last sas_reduce_radial on this context. */
sas_status sas_get_reduce_time(sas_ctx* ctx, double* ms);

const char* sas_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SAS_H */
