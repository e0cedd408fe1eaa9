/* =====================================================================================
 * xt.h -- C ABI of the B200-native multi-turn single-particle tracking engine.
 *
 * What the library computes.  "The beam line is represented as a sequence of ... objects
 * ..., each corresponding to an accelerator element" (section "Lattice
 * modelling and single particle tracking"); "a 'thin' lattice integration method is
 * adopted"; one compiled kernel is "able to track the entire beamline"
 * for "particles ensembles"; aperture elements "check the
 * particle positions with respect to the defined aperture and stop the tracking for the
 * particles found to be outside"; particles are independent on
 * non-collective lines.  The paper prints no map formulas; the maps are
 * those fixed in DESIGN.md section 5 (canonical arithmetic order included).
 *
 * Conventions.  Plain pointers and sizes only.  Every particle pointer is a DEVICE pointer
 * unless the function name ends in _host.  All calls that take a stream are asynchronous on
 * that stream and never synchronise the host (the _host variants do, once, at the end).
 * Return value: 0 (XT_OK) or a negative xt_status; on failure no output is written and
 * xt_last_error() holds a thread-local message.  No exceptions, no abort().
 * There is no CPU fallback: without a CUDA device every compute entry point fails with
 * XT_ERR_CUDA.
 * ===================================================================================== */
#ifndef XT_H_
#define XT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  XT_OK = 0,
  XT_ERR_INVALID_ARG = -1, /* NULL pointer, negative count, bad option                       */
  XT_ERR_BAD_LATTICE = -2, /* bad magic/version/size, unknown type, truncated buffer,         */
                           /* order > XT_MAX_ORDER, non-finite parameter, p0c/mass0 <= 0      */
  XT_ERR_CUDA = -3,        /* CUDA runtime failure (message in xt_last_error)                 */
  XT_ERR_NOMEM = -4,       /* host or device allocation failed                                */
  XT_ERR_UNSTABLE = -5     /* xt_twiss4d: probe particle lost, singular map or no convergence  */
} xt_status;

#define XT_MAX_ORDER 20

/* Element type ids of the packed lattice buffer (magnets, cavities, aperture
 * restrictions; tilts / misalignments as changes of the reference system). */
enum {
  XT_MARKER = 0,
  XT_DRIFT = 1,       /* length                                                  (map M1)   */
  XT_MULTIPOLE = 2,   /* aux = order N; hxl, length, knl[0..N], ksl[0..N] (raw)  (map M2)   */
  XT_CAVITY = 3,      /* voltage [V], frequency [Hz], lag [deg]                  (map M3)   */
  XT_SROTATION = 4,   /* cos_z, sin_z                                            (map M4)   */
  XT_XYSHIFT = 5,     /* dx, dy                                                  (map M4)   */
  XT_LIMITRECT = 6,   /* min_x, max_x, min_y, max_y (edges inclusive)            (step A)   */
  XT_LIMITELLIPSE = 7,/* a, b (edge inclusive)                                   (step A)   */
  XT_QUADRUPOLE = 8,  /* k1 [1/m^2], length [m]: thick quadrupole, k1 != 0, length > 0           */
                      /* (reading A18)             */
  XT_BEND = 9,        /* k0 [1/m], h [1/m], length [m]: thick sector bend, k0*h > 0, length > 0; */
                      /* aux = 0: the 'expanded' map (reading A19), aux = 1: the 'full' */
                      /* map, the exact helix in the uniform field (reading A23)    */
  XT_LIMITPOLYGON = 10,/* aux = n vertices (3..256); x[0..n), y[0..n): closed polygon, even-odd   */
                      /* rule, NaN lost ("polygonal"; reading A20)         */
                      /* 11 is reserved (internal)                                                */
  XT_RADMULTIPOLE = 12/* parameters as XT_MULTIPOLE, length > 0: thin multipole with "mean"       */
                      /* synchrotron radiation (reading A22)              */
};

/* Packed lattice buffer (HOST memory, little-endian, 8-byte aligned records):
 *   header, 48 B: char magic[8] = "XTLAT001"; uint32 version = 1; uint32 n_elements;
 *                 double p0c [eV]; double mass0 [eV]; double q0 [e]; uint64 total_bytes
 *   n_elements records: uint32 type; uint32 aux; double params[...] as listed above.
 * beta0, gamma0 are derived inside: E0 = sqrt(p0c^2 + mass0^2), beta0 = p0c/E0,
 * gamma0 = E0/mass0.  Multipole strengths follow the MAD-X convention (PAPER.md:70,
 * "imported from MAD-X"): knl[n] = integrated d^n By/dx^n / (P0/q0), NOT divided by n!. */

typedef struct xt_lattice xt_lattice; /* opaque; immutable after create; owns its device image */

/* Particle ensemble, structure of arrays, each of length n_part, caller-owned.
 * x, y, zeta [m]; px = Px/P0, py = Py/P0; delta = (P-P0)/P0; ptau = (E-E0)/(P0 c);
 * rpp = P0/P; rvv = beta/beta0.  delta AND ptau are both state (reading A7): they
 * are loaded and stored verbatim so that n calls of k turns equal one call of n*k turns
 * bit for bit.  state: 1 alive, 0 lost on an aperture.  For a lost particle the coordinates
 * are those AT the aperture that stopped it, at_element is that element's index in the
 * packed buffer, s the sum of drift and thick-element lengths before it, at_turn the number of COMPLETED
 * turns.  For survivors s = 0 and at_turn has advanced by n_turns.
 * particle_id and at_element may be NULL.  particle_id is never written. */
typedef struct {
  double *x, *px, *y, *py, *zeta, *delta;
  double *ptau, *rpp, *rvv;
  double *s;
  int64_t *at_turn, *state;
  int64_t *particle_id, *at_element;
} xt_particles;

/* Timing record of one xt_track_ex call (optional, HOST memory).  Asking for it makes the call
 * synchronous: it brackets every tracking launch and every compaction pass (step C: count, scan, move)
 * with CUDA events on the stream, synchronises at the end and fills the record.  Algorithmic bytes of a
 * pass over n_in particles: 2 x n_in x 112 B (every one of the 13 arrays and the
 * origin index is read once and written once, to the next working set or to its final place). */
#define XT_STATS_MAX_PASSES 128
typedef struct {
  int64_t n_track_launches;   /* tracking launches of the call                                   */
  int64_t n_passes;           /* compaction passes, the initial partition included (0: none ran) */
  double track_ms;            /* sum of the tracking launches' device times                      */
  double compact_ms;          /* sum of the passes' device times                                 */
  double compact_bytes;       /* sum of their algorithmic bytes                                  */
  double scatter_ms;          /* the final restore-order scatter                                 */
  double scatter_bytes;       /* 2 x n_alive x 112                                               */
  int64_t pass_n_in[XT_STATS_MAX_PASSES];   /* particles entering pass k (first passes only)     */
  int64_t pass_n_out[XT_STATS_MAX_PASSES];  /* alive behind it                                   */
  double pass_ms[XT_STATS_MAX_PASSES];
} xt_track_stats;

/* Options of xt_track_ex.  Zero-initialise for the defaults. */
typedef struct {
  int64_t turns_per_launch; /* 0: auto (= compact_every when compaction is active, else all)  */
  int64_t compact_every;    /* 0: auto (1000 turns if the lattice has apertures and n_turns   */
                            /*    exceeds it); < 0: never compact; > 0: period in turns       */
  int32_t block_size;       /* 0: auto; else threads per CTA, a multiple of 32 in [32, 256]   */
  int32_t particles_per_thread; /* 0: auto; else 1, 2, 3 or 4                                 */
  void *workspace;          /* DEVICE scratch for compaction, caller-owned, or NULL: the      */
  uint64_t workspace_bytes; /*    library then uses cudaMallocAsync / cudaFreeAsync on the    */
                            /*    stream.  xt_track_workspace_bytes(n_part) bytes, 256-byte   */
                            /*    aligned; too small for step C: XT_ERR_INVALID_ARG.  With it */
                            /*    xt_track_ex allocates nothing.                              */
  xt_track_stats *stats;    /* HOST, optional: see xt_track_stats (makes the call synchronous) */
  int32_t cold_in_registers;/* 0: auto; 1: keep the per-particle functions of (delta, ptau) in   */
                            /*    registers; -1: in shared                                         */
                            /*    memory.                                                        */
                            /*    Launch-shape option like the two above: results are            */
                            /*    bit-identical for every shape.                                 */
  int32_t balance;          /* launch shapes with the cold state in registers (the auto shapes  */
                            /*    up to ~2 million particles):                                  */
                            /*    0: auto, -1: never, 1: always, n > 1: always, n turns per item. */
                            /*    The launch has one CTA per (group of particles, block of      */
                            /*    turns) item and a queue of ready groups in device memory, so    */
                            /*    that an ensemble that does not fill a whole number of CTAs per  */
                            /*    SM still keeps every SM busy with full warps (DESIGN.md section */
                            /*    6.2b).  Needs 4 bytes per item + 16: from `workspace` when      */
                            /*    given, else stream-ordered.  Launch-shape option: bit-identical */
                            /*    results.  > 0 with a shape that keeps the cold state in shared  */
                            /*    memory: XT_ERR_INVALID_ARG.                                     */
} xt_track_opts;

/* Static description of a lattice image; counts are per turn. */
typedef struct {
  int64_t n_elements;       /* records in the packed buffer (markers included)                */
  int64_t n_records;        /* records in the device image (markers dropped)                  */
  int64_t n_chunks;         /* TMA chunks per turn                                            */
  int64_t image_bytes;      /* bytes of the device image                                      */
  int64_t chunk_bytes;      /* shared-memory bytes of one staging buffer                      */
  int64_t n_by_type[8];     /* elements per XT_* type id                                      */
  int64_t sum_order;        /* sum of N over all multipoles                                   */
  int64_t n_curved;         /* multipoles with hxl != 0                                       */
  int64_t has_aperture;     /* 1 if any LimitRect / LimitEllipse / LimitPolygon               */
  double beta0, gamma0;     /* reference particle as derived by the packer                    */
  double circumference;     /* sum of drift and thick-element lengths [m]                     */
  int64_t n_drift_evals;    /* sqrt evaluations per turn after fusion (consecutive drifts     */
                            /* share one; equals the number of drifts when fuse is off)       */
  int64_t n_thick;          /* thick elements (XT_QUADRUPOLE, XT_BEND); not in n_by_type      */
  int64_t n_drift_applies;  /* drift applications per turn: the number of drifts, minus what   */
                            /* the production build saves by applying consecutive drifts as    */
                            /* one drift of the summed length (exact composition; the          */
                            /* validation build applies every drift)                           */
} xt_lattice_info;

/* Options of xt_lattice_create_ex.  Zero-initialise for the defaults.  Neither changes any
 * result: the same maps run in the same order with the same arithmetic. */
typedef struct {
  int64_t chunk_bytes; /* 0: default (8192);  else shared-memory bytes of one staging buffer,  */
                       /*    a multiple of 128 in [1024, 65536], at least one record + 16      */
  int32_t fuse;        /* 0 or 1: [Drift] Multipole [Drift] share one record and one dispatch; */
                       /*    2: one record per element                                         */
  int32_t reserved;
} xt_lattice_opts;

/* Step P: parse + validate the packed buffer, pre-scale the multipole
 * coefficients, fold curvature into the dipole term, lay out 16-byte-aligned records in
 * Horner order, cut them into TMA chunks and copy the image to the current CUDA device.
 * The caller may free `packed` as soon as the call returns.  *out untouched on failure. */
int xt_lattice_create(const void *packed, size_t nbytes, xt_lattice **out);
int xt_lattice_create_ex(const void *packed, size_t nbytes, const xt_lattice_opts *opts,
                         xt_lattice **out);
int xt_lattice_destroy(xt_lattice *lat);
int xt_lattice_get_info(const xt_lattice *lat, xt_lattice_info *info);
/* s position (entrance) of every element; `out` is a HOST array of `cap` doubles; returns
 * n_elements (>= 0) or a negative xt_status. */
int64_t xt_lattice_s_table(const xt_lattice *lat, double *out, int64_t cap);

/* Host-only form of step P for tests and tools (makes NO CUDA call): packs the image exactly
 * as xt_lattice_create_ex would upload it.  Copies min(image size, cap) bytes to `image` (HOST;
 * may be NULL when cap == 0), fills *info if non-NULL, returns the image size in bytes or a
 * negative xt_status. */
int64_t xt_lattice_pack_host(const void *packed, size_t nbytes, const xt_lattice_opts *opts,
                             void *image, size_t cap, xt_lattice_info *info);

/* Steps L, S, D, M1-M4, A, T, W (+ C when compaction is active): track every particle with
 * state == 1 for n_turns turns through the whole line.  DEVICE pointers.
 * On (stream-ordered) return the arrays are in their ORIGINAL order even if the alive
 * particles were compacted internally.  n_part == 0 or n_turns == 0 is a successful no-op.
 * Calling it again continues the run. */
int xt_track(const xt_lattice *lat, const xt_particles *p, int64_t n_part, int64_t n_turns,
             void *cuda_stream);
int xt_track_ex(const xt_lattice *lat, const xt_particles *p, int64_t n_part, int64_t n_turns,
                void *cuda_stream, const xt_track_opts *opts);

/* Bytes of device scratch for n_part particles: what step C needs (two working sets of 14 arrays, tile
 * counts, two counters) and, behind it, the queue of the balanced mode for the auto launch shapes.
 * xt_track_opts.workspace should provide this much; one that only holds step C's part is accepted and
 * the balanced mode is then not used with compaction. */
uint64_t xt_track_workspace_bytes(int64_t n_part);

/* xt_track_ex for callers that cannot allocate (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): the same steps with the same results (bit-identical to
 * xt_track_ex in the same build), but the scratch of step C (particles stopped by
 * an aperture are retired, the alive ones packed) is a fixed array in the library's device image
 * instead of a stream-ordered allocation.  The call makes no cudaMalloc / cudaFree /
 * cudaMallocAsync and calls no allocating library routine.
 *   - n_part <= XT_TRACK_STATIC_MAX_PARTICLES, else XT_ERR_INVALID_ARG (xt_last_error names the
 *     limit).  The array is 7.0 MiB (the working sets of step C for the limit); every GPU that
 *     loads the library holds it until the process exits.
 *   - opts may be NULL; opts->workspace, ->workspace_bytes and ->stats must be 0 / NULL (the
 *     stats record creates events and allocates): XT_ERR_INVALID_ARG otherwise.
 *   - p: DEVICE arrays, the caller's inputs and outputs as in xt_track_ex; nothing else is kept.
 *   - ALL calls on a device share the one array, which keeps the previous call's bytes (the
 *     call clears what must start at zero itself).  Two xt_track_static calls whose GPU work can
 *     overlap (different streams, or graphs launched concurrently) RACE on it: order them on one
 *     stream or with events.  Calls on different devices do not interact.
 *   - Runs without compaction use at most the first bytes of it (the queue of the balanced mode,
 *     xt_track_opts.balance) or nothing at all.  With compaction the queue only fits behind the
 *     working sets of smaller ensembles: otherwise the balanced mode is not used (balance > 0:
 *     XT_ERR_INVALID_ARG). */
#define XT_TRACK_STATIC_MAX_PARTICLES 32768
int xt_track_static(const xt_lattice *lat, const xt_particles *p, int64_t n_part, int64_t n_turns,
                    void *cuda_stream, const xt_track_opts *opts);

/* End-to-end variant: the SAME call with HOST arrays.  Copies the ensemble to the device
 * (stream-ordered allocation), tracks, copies everything back and synchronises the stream.
 * Pinned host memory makes the copies asynchronous; pageable memory also works. */
int xt_track_host(const xt_lattice *lat, const xt_particles *host_p, int64_t n_part,
                  int64_t n_turns, void *cuda_stream, const xt_track_opts *opts);

/* Init helper: delta -> ptau, rpp, rvv for n particles (DEVICE). */
int xt_particles_init_derived(const xt_lattice *lat, const xt_particles *p, int64_t n_part,
                              void *cuda_stream);

/* Step H: survival-turn histogram (BASELINE.json configs[4]).  hist (DEVICE, int64[n_bins+1])
 * is OVERWRITTEN: hist[b] = #{state == 0 and bin_width*b <= at_turn < bin_width*(b+1)},
 * lost particles with at_turn beyond the last bin go to bin n_bins-1, and
 * hist[n_bins] = #{state == 1} (survivors). */
int xt_survival_histogram(const int64_t *at_turn, const int64_t *state, int64_t n_part,
                          int64_t bin_width, int64_t n_bins, int64_t *hist, void *cuda_stream);

/* FP64 FMA microbenchmark (roofline denominator, north_star: "measured by an FMA
 * microbenchmark in the same run"): runs register-resident DFMA kernels on the whole chip -- a sweep
 * over operand forms (fma(acc, a, b) with a, b kernel parameters; one per-chain vector register plus
 * one parameter as multiplicand or as addend), 4-16 independent chains per thread and launch shapes of
 * 128-1024 threads x 1-4 CTAs per SM -- times each with CUDA events on `cuda_stream`, synchronises,
 * and returns the MAXIMUM in FLOP/s (2 per FMA) in *flops_per_s and that kernel's time in *ms (either
 * may be NULL).  On B200 the maximum is 2.00 cycles per warp DFMA per scheduler. */
int xt_fp64_fma_peak(double *flops_per_s, double *ms, void *cuda_stream);
/* One row of that sweep: shape `index` in [0, xt_fp64_fma_peak_sweep_size()); desc (HOST, 4 ints, may be
 * NULL) receives {chains per thread, operand form 0/1/2, threads per CTA, CTAs per SM}.
 * XT_ERR_INVALID_ARG for an index out of range. */
int xt_fp64_fma_peak_sweep_size(void);
int xt_fp64_fma_peak_sweep(int index, double *flops_per_s, double *ms, int *desc, void *cuda_stream);
/* The same measurement with the operand shapes of the tracking arithmetic:
 * pattern 0 = xt_fp64_fma_peak; 1 = three distinct vector-register operands per DFMA; 2 = the complex
 * Horner recurrence of step M2 for 4 particles per thread, coefficients broadcast from shared memory,
 * no lattice; 3 = the same recurrence with the coefficients in uniform registers (constant memory). */
int xt_fp64_fma_probe(int pattern, double *flops_per_s, double *ms, void *cuda_stream);

/* Twiss from tracking, 4-D ("Twiss module"): the closed
 * orbit at the start of the line for momentum deviation delta0 (zeta = 0) by Newton iteration on
 * the one-turn map (step 1), the 4x4 one-turn Jacobian there by central differences of tracked
 * particles (step 2; steps 1e-6 m / 1e-8 rad), and the uncoupled linear optics per plane (step 3:
 * cos mu = (M11+M22)/2, beta = M12/sin mu, alpha = (M11-M22)/(2 sin mu)).  Every Newton step is one
 * xt_track launch of nine particles through the whole line; only the 4x4 algebra is host code.
 * guess4 (HOST, x px y py; may be NULL = origin).  Synchronises the stream.  XT_ERR_UNSTABLE if a
 * probe particle is lost, M - 1 is singular, or 25 steps do not reach |dz| < 1e-13; an unstable
 * plane (|cos mu| >= 1) is reported through stable = 0 and NaN optics, not as an error.
 * Limitation of the 4-D entry points (xt_twiss4d, _chrom, _line): the probes are tracked through the line
 * AS IT IS, live RF cavities included.  They start at zeta = 0 but slip before they reach a cavity and pick
 * up a small energy kick there, so in a ring with cavities on, the "4-D" orbit, dispersion and chromaticity
 * contain that longitudinal motion (relative 1e-4 on the dispersion downstream of the cavities of the
 * LHC-sized configs).  Pass a lattice without cavities for a pure 4-D result, or use xt_twiss6d.  The oracle
 * procedure (oracle/make_optics.py) tracks the same way, so parity does not see this. */
typedef struct {
  double co[4];                 /* closed orbit x, px, y, py                                    */
  double m[16];                 /* one-turn Jacobian at the closed orbit, row-major              */
  double betx, alfx, mux, qx_frac; /* mu in rad in (-pi, pi], q = mu/2pi mod 1                    */
  double bety, alfy, muy, qy_frac;
  int32_t iterations, stable;
} xt_twiss4d_result;
int xt_twiss4d(const xt_lattice *lat, double delta0, const double *guess4, xt_twiss4d_result *out,
               void *cuda_stream);

/* Loss-location refinement ("particle backtracking and a locally
 * refined aperture model obtained by polygonal interpolation", Fig. 4; reading A20 and
 * section 16).  For every particle of `p` (DEVICE, as left by xt_track on `lat`) with state == 0 whose
 * at_element is a LimitRect / LimitEllipse / LimitPolygon with length between it and the previous aperture (or
 * the start of the line): the particle is tracked back to that upstream aperture and forward again in
 * steps of at most `ds` [m] through polygons of `n_poly` vertices (3..256) interpolated between the
 * two apertures, shifts and tilts included; x, px, y, py, zeta, delta, ptau, rpp, rvv and s are
 * overwritten with the values at the first polygon it fails (s = position of that polygon); state,
 * at_turn and at_element are kept.  A particle that fails none keeps its record.  All tracking runs in
 * the xt_track kernels on small lattices built on the host from the packed buffer the lattice was
 * created from; one pair of launches per flagging aperture.  p->at_element must not be NULL.  Call it
 * once per tracked ensemble: a refined record no longer sits at its at_element.
 * *n_refined (HOST, may be NULL) = number of records moved.  Synchronises the stream. */
int xt_refine_loss_location(const xt_lattice *lat, const xt_particles *p, int64_t n_part, double ds,
                            int32_t n_poly, int64_t *n_refined, void *cuda_stream);

/* Time functions ("time dependent knobs that are updated automatically
 * during the simulation", Fig. 1; PAPER.md:80 one parameter controlling groups of elements; DESIGN.md reading
 * A21 and section 17).  Time advances in turns.  `table` (HOST, row-major [n_knobs][n_steps]) holds the knob
 * values f_k[step]; a link adds gain * f_knob[step] to knl[order] (skew = 0) or ksl[order] (skew = 1) of the
 * XT_MULTIPOLE with index `element` in the packed buffer: value = base, then value = value + gain * f for the
 * links of that coefficient in the order given (product rounded, then the sum); what the packer derives from
 * the coefficient follows (knl/n!, the curvature fold, the weak-focusing term).  The call copies table and
 * links to the device and replaces any earlier set; n_links == 0 removes it.  XT_ERR_BAD_LATTICE if a link
 * does not name a multipole coefficient that exists or a knob of the table.  A call that fails leaves the
 * lattice with the knob set it had. */
typedef struct {
  int64_t element;
  int32_t order, skew, knob, reserved;
  double gain;
} xt_knob_link;
int xt_lattice_set_knobs(xt_lattice *lat, const double *table, int32_t n_knobs, int64_t n_steps,
                         const xt_knob_link *links, int64_t n_links);
/* xt_track for n_turns turns with the knobs applied: before turn j (0-based) a small kernel rewrites the linked
 * coefficients in the device image for step = clamp(step0 + j, 0, n_steps - 1), then the tracking kernel runs
 * that turn (one launch per turn, stream-ordered, no host synchronisation); afterwards the image is back at
 * its base values.  The lattice is NOT const here: the call rewrites its device image in place, so while it
 * runs the lattice must not be used by another stream or thread.  No loss compaction. */
int xt_track_knobs(xt_lattice *lat, const xt_particles *p, int64_t n_part, int64_t n_turns,
                   int64_t step0, void *cuda_stream);

/* Dispersion and chromaticity at the start of the line ("tunes, beta, alpha,
 * dispersion"): xt_twiss4d at delta0 and at delta0 -+ ddelta (ddelta > 0, e.g. 1e-4; the
 * off-momentum searches start from the on-momentum orbit); dispersion = central difference of the closed
 * orbit, chromaticity = central difference of the fractional tunes taken on the circle.  Errors as
 * xt_twiss4d; NaN chromaticity in a plane that is unstable at any of the three momenta. */
typedef struct {
  xt_twiss4d_result on;    /* at delta0                                                       */
  double dx, dpx, dy, dpy; /* d(closed orbit)/d(delta)                                        */
  double dqx, dqy;         /* d(tune)/d(delta)                                                */
} xt_twiss4d_chrom_result;
int xt_twiss4d_chrom(const xt_lattice *lat, double delta0, double ddelta, const double *guess4,
                     xt_twiss4d_chrom_result *out, void *cuda_stream);

/* Twiss steps 1-3 in six dimensions for a ring with an RF cavity ("6x6 Jacobian by
 * central differences (13 particles through xt_track)"): Newton on (x, px, y, py, zeta, delta)
 * with one launch of thirteen probes per step (steps 1e-6 m, 1e-8, 1e-6 m, 1e-8, 1e-5 m, 1e-8), the 6x6
 * Jacobian at the fixed point, and the three tunes from its reciprocal characteristic polynomial: with
 * u = lambda + 1/lambda the cubic u^3 - s1 u^2 + s2 u - s3 = 0 (s1 = e1, s2 = e2 - 3, s3 = e3 - 2 e1, e_k the
 * elementary symmetric functions from the traces of M, M^2, M^3) has the roots 2 cos mu_k.  qs = the smallest
 * angle / 2 pi, in (0, 1/2); q1 (q2) = the remaining one closer to the horizontal (vertical) 2x2 block, its side
 * of the half integer from the sign of that block's M12.  guess6 (HOST, may be NULL = origin).
 * XT_ERR_UNSTABLE: probe lost, no convergence in 25 steps, M - 1 singular (no cavity), or a root outside
 * (-2, 2).  Synchronises the stream. */
typedef struct {
  double co[6];  /* x, px, y, py, zeta, delta */
  double m[36];  /* row-major, in these variables */
  double q1_frac, q2_frac, qs;
  int32_t iterations, reserved;
} xt_twiss6d_result;
int xt_twiss6d(const xt_lattice *lat, const double *guess6, xt_twiss6d_result *out, void *cuda_stream);

/* Linear normal form in six dimensions (Twiss steps 3-5).  Pure HOST
 * arithmetic, no CUDA call.  m: the 6x6 one-turn matrix of xt_twiss6d_result (row-major, variables x, px, y,
 * py, zeta, delta); rvv_co = beta/beta0 on the closed orbit, which turns delta into the canonical
 * pzeta = ptau/beta0 (d pzeta = rvv d delta; 1 for delta = 0).  The three pairs of eigenvalues follow from the
 * cubic of xt_twiss6d; the eigenvector of exp(i mu_k) is (M - conj(lambda_k)) prod_{j != k} (M^2 - u_j M + 1) w;
 * of each conjugate pair the one with v^H S v = +2i is kept.  Mode 3 is the one with the smallest tune angle
 * (longitudinal); of the other two, mode 1 has the larger horizontal part; phase origin: the mode's own plane
 * (x, y, zeta) real positive.  bet[u][k], alf[u][k]: Mais-Ripken functions of mode k in plane u (0 x, 1 y,
 * 2 zeta): |v_u|^2 and -Re(conj(v_u) v_pu).  disp: dispersion "from the eigenvectors", Re(v_u / v_pzeta) of
 * the longitudinal mode per unit delta (dx, dpx, dy, dpy).  q_frac[k]: arg(lambda_k)/2 pi in [0, 1).
 * stable = 0 (and NaN) if an eigenvalue leaves the unit circle; degenerate = 1 (and NaN) if two modes have the
 * same tune within what a central-difference matrix resolves. */
typedef struct {
  double q_frac[3];
  double bet[3][3], alf[3][3]; /* [plane][mode] */
  double disp[4];
  double v[3][12];             /* eigenvectors: (re, im) of x, px, y, py, zeta, pzeta */
  int32_t stable, degenerate;
} xt_twiss6d_modes;
int xt_twiss6d_normal_form(const double *m, double rvv_co, xt_twiss6d_modes *out);

/* The six-dimensional optics along the line (the eigenvectors are propagated "to all other
 * elements by tracking").  xt_twiss6d at the start, its normal form, then ONE launch of thirteen probes (the
 * closed orbit and +-h along the six coordinates) through a copy of the line with a monitor record in front of
 * every element; per row the host forms the 6x6 Jacobian from the start (canonical variables at both ends) and
 * carries the three eigenvectors through it.  rows (HOST, cap >= n_elements + 1): row i = the entrance of
 * element i, the last row the end of the line.  mu[k]: phase of mode k's own component from the start,
 * unwrapped (the betatron phases only grow; the synchrotron phase is counted in its own sense).  start,
 * start_modes may be NULL.  Errors as xt_twiss6d; XT_ERR_UNSTABLE also for degenerate modes.  Synchronises. */
typedef struct {
  double s;
  double co[6];                /* closed orbit: x, px, y, py, zeta, delta */
  double bet[3][3], alf[3][3]; /* [plane][mode] */
  double mu[3];
  double disp[4];              /* dx, dpx, dy, dpy per unit delta, from the longitudinal eigenvector */
} xt_twiss6d_row;
int xt_twiss6d_line(const xt_lattice *lat, const double *guess6, xt_twiss6d_result *start,
                    xt_twiss6d_modes *start_modes, xt_twiss6d_row *rows, int64_t cap, void *cuda_stream);

/* Linear normal form of a 4x4 one-turn matrix with coupling (PAPER.md:98 step 3 "from the eigenvalues and
 * eigenvectors of the Jacobian matrix", step 5 "Mais-Ripken").  Pure HOST arithmetic,
 * no CUDA call.  m: row-major, e.g. xt_twiss4d_result.m.  The characteristic polynomial of a symplectic
 * matrix is reciprocal: with u = lambda + 1/lambda it is u^2 - tr(M) u + (tr(M)^2 - tr(M^2))/2 - 2 = 0, so
 * cos mu_k = u_k/2; the eigenvector of exp(i mu_k) is (M - conj(lambda_k)) (M^2 - u_other M + 1) w; of each
 * conjugate pair the one with v^H S v = +2i is kept (in one uncoupled plane: (sqrt(beta),
 * (i - alpha)/sqrt(beta)), eigenvalue exp(+i mu)); mode 1 is the one with the larger horizontal part, its x
 * component real positive (mode 2: y).  beta_uk = |v_u|^2, alpha_uk = -Re(conj(v_u) v_pu).
 * stable = 0 (and NaN) if an eigenvalue leaves the unit circle; degenerate = 1 (and NaN) if the two modes have
 * the same tune (|cos mu_1 - cos mu_2| < 1.6e-4, what a central-difference Jacobian resolves): the eigenvectors
 * are then not defined (use the per-plane optics). */
typedef struct {
  double q1_frac, q2_frac;
  double betx1, alfx1, bety1, alfy1;
  double betx2, alfx2, bety2, alfy2;
  double v1[8], v2[8]; /* eigenvectors (x, px, y, py), re/im interleaved */
  int32_t stable, degenerate;
} xt_twiss4d_modes;
int xt_twiss4d_normal_form(const double *m, xt_twiss4d_modes *out);

/* Optics along the line (the optics found at the start is carried
 * "to all other elements by tracking"; beta functions along the ring).  After the three closed-orbit
 * searches of xt_twiss4d_chrom, ONE launch tracks eleven probe particles (the orbit, +-h along x, px, y, py,
 * and the closed orbits at delta0 -+ ddelta) through the line with an internal monitor record in front of
 * every element; from the rows the host forms, per element entrance, the closed orbit, the 4x4 Jacobian
 * J_i from the start by central differences, per plane beta_i = m11^2 b0 - 2 m11 m12 a0 + m12^2 g0,
 * alpha_i = -m11 m21 b0 + (m11 m22 + m12 m21) a0 - m12 m22 g0, mu_i = atan2(m12, m11 b0 - m12 a0) unwrapped
 * along the line (mux of the last row / 2 pi is the tune WITH its integer part), and the dispersion as the
 * central difference of the two off-momentum orbits.  rows: HOST array of cap >= n_elements + 1 entries;
 * row i is the entrance of element i, row n_elements the end of the line.  start may be NULL.  Errors as
 * xt_twiss4d (XT_ERR_UNSTABLE also if a probe is lost on the way or a plane is unstable). */
typedef struct {
  double s, x, px, y, py;
  double betx, alfx, mux, bety, alfy, muy;
  double dx, dpx, dy, dpy;
  double betx1, bety1, betx2, bety2; /* Mais-Ripken beta functions of the two normal modes (xt_twiss4d_normal_form) */
  double mu1, mu2;                   /* their phase advances from the start, unwrapped; NaN like the four above  */
                                     /* when the one-turn matrix has no two distinct stable modes                */
} xt_twiss_row;
int xt_twiss4d_line(const xt_lattice *lat, double delta0, double ddelta, const double *guess4,
                    xt_twiss4d_chrom_result *start, xt_twiss_row *rows, int64_t cap, void *cuda_stream);

/* Number of kernels the library has launched from this process so far (bench bookkeeping). */
int64_t xt_launch_count(void);

const char *xt_last_error(void); /* thread-local, never NULL */
const char *xt_build_info(void); /* e.g. "sm_100a fmad=true" / "sm_100a fmad=false"          */

#ifdef __cplusplus
}
#endif
#endif /* XT_H_ */
