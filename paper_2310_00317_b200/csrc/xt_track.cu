// The tracking kernel for sm_100a.
//
// "Xtrack ... assembles and compiles a C kernel ... able to track the entire beamline"
// (PAPER.md:74): here that kernel is hand-written and interprets a packed record stream.
// One thread owns P particles (P = 1..4, interleaved so that every global access is
// coalesced) and keeps their hot state (x, px, y, py, zeta) in registers across all elements
// and turns; SoA FP64 loads/stores happen only at the start and end of the launch (and, for a
// particle that hits an aperture, once at the moment it is lost).  The lattice image is
// streamed chunk by chunk from L2 into shared memory with 1-D TMA bulk copies
// (cp.async.bulk + mbarrier complete_tx), double-buffered; every thread of the CTA reads the
// same record, so each LDS.128 is a broadcast.  Dispatch is a switch on a value all lanes
// share (warp-uniform); a record is usually a fused [drift] kick [drift] group
// (xt_internal.h).  Multipoles are a complex Horner recurrence of FMAs.
//
// Instantiations xt_track_kernel<P, THICK, REG, NFIX>: P particles per thread; THICK = the extended
// maps (thick elements, polygons, radiation, monitors) compiled in; REG = the cold per-particle state
// (functions of delta, ptau) in registers instead of shared memory (small ensembles); NFIX = 15: the
// handlers of order-15 multipoles fully unrolled (lattices the packer finds full of them).
//
// Why P > 1 (profiles/r01b_track_p1_summary.md): with one particle per thread 58 % of the
// issued warp instructions were not FP64 (dispatch, LDS, branches, the slow-path guards of
// sqrt and /) and the FP64 pipe sat at 49 %.  P particles per thread share every one of those
// instructions and give each warp P independent FP64 chains.
//
// What bounds it (profiles/r02_dfma_peak_sweep.md): an FP64 instruction costs max(2, number of
// vector-register source operands) cycles of its scheduler's FP64 pipe, and nearly every DFMA of this
// arithmetic has three (re x + t; x += px lpz; c - im y with c loaded from shared memory).
//
// Arithmetic.  The maps are written in the canonical order of DESIGN.md section 5 through
// XT_MADD / XT_NMADD / XT_MUL.  The validation build (--fmad=false, XT_FMAD_OFF) evaluates
// exactly those trees with IEEE sqrt and division and is bit-identical to the oracle on
// cavity-free lattices.  The production build fuses every a*b + c into one DFMA (explicitly,
// so that results do not depend on the launch shape), replaces the drift's sqrt + division
// by branch-free Newton sequences on the MUFU.RSQ64H / MUFU.RCP64H seeds (DESIGN.md section
// 6.3: same formula, <= 2 ulp on the increments) and receives consecutive drifts merged into one
// (xt_lattice.cu pass 1b); the measured distance to the oracle is set by FMA fusion (<= 0.2 of the
// 1e-12 bar in x, y; 0.03 in zeta).
#include <atomic>

#include "xt_internal.h"

namespace xt {
namespace {

// Balanced mode: turns in the first item of group g.  The later items have block_turns turns each; the first
// ones are staggered (1 .. block_turns, by a hash of the group) so that the CTAs of one SM do not all finish,
// wait and restart at the same moments -- the load only evens out when their waits do not coincide.
__host__ __device__ inline int64_t first_block_turns(uint32_t group, int64_t block_turns) {
  return 1 + static_cast<int64_t>(((group * 2654435761u) >> 8) % static_cast<uint32_t>(block_turns));
}

struct TrackArgs {
  const unsigned char *image;
  const ChunkDesc *chunks;
  const double *s_table;
  const int64_t *n_active;  // device counter (compaction path) or nullptr
  double *monitor_rows;     // where TAG_MON records store (xt_twiss4d_line), else nullptr
  xt_particles p;
  int64_t n_part;
  int64_t n_turns;
  int32_t n_chunks;
  uint32_t chunk_bytes;
  int32_t stage_chunks;  // consecutive chunks staged by one bulk copy (they are contiguous in the image)
  int32_t grid_quantum;  // CTAs are handed out in multiples of this (the SM count)
  double beta0, tib, igam2;
  // Balanced mode (cold-state-in-registers shapes only; nullptr otherwise): the CTAs are persistent and
  // draw (group of particles, block of turns) items from a first-in first-out queue.  queue[0]: pop
  // tickets; queue[1]: pushes; queue[2]: finished groups; queue[4 + n]: item of push n, plus one.
  unsigned int *queue;
  int32_t block_turns;  // turns per item (the first item of a group: first_block_turns)
};

__device__ __forceinline__ uint32_t smem_addr(const void *p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}

// Arm the barrier with the byte count and start the bulk copy global -> shared (TMA, 1-D).
__device__ __forceinline__ void tma_load_chunk(uint32_t bar, uint32_t dst, const void *src, uint32_t bytes) {
  // order earlier generic-proxy reads of the buffer before the async-proxy overwrite
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
      "l"(src), "r"(bytes), "r"(bar)
      : "memory");
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "XT_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra XT_DONE_%=;\n"
      "bra XT_WAIT_%=;\n"
      "XT_DONE_%=:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}

// a*b + c and c - a*b.  The validation build rounds the product and the sum separately, as
// the oracle does; the production build fuses them, explicitly, so that the arithmetic does
// not depend on which contractions the compiler happens to pick in each instantiation
// (results are bit-identical for every launch shape).  XT_MUL is a product that is never
// fused into a neighbouring sum.
#ifdef XT_FMAD_OFF
#define XT_MADD(a, b, c) ((a) * (b) + (c))
#define XT_NMADD(a, b, c) ((c) - (a) * (b))
#else
#define XT_MADD(a, b, c) fma((a), (b), (c))
#define XT_NMADD(a, b, c) fma(-(a), (b), (c))
#endif
#define XT_MUL(a, b) __dmul_rn((a), (b))

// XT_CANONICAL_DRIFT: IEEE sqrt and division in the canonical order of DESIGN.md section 5
// (always in the validation build; -DXT_CANONICAL_DRIFT gives a production build with them).
#if defined(XT_FMAD_OFF) && !defined(XT_CANONICAL_DRIFT)
#define XT_CANONICAL_DRIFT
#endif

#ifndef XT_CANONICAL_DRIFT
// MUFU.RSQ64H / MUFU.RCP64H: ~20-bit seeds computed from the high word of the operand.
__device__ __forceinline__ double rsqrt_seed(double a) {
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
  return r;
}
__device__ __forceinline__ double rcp_seed(double a) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
  return r;
}
#endif

constexpr int kPrefetch = 4;  // 16-byte slots of a record loaded ahead of its dispatch ...
#ifndef XT_PF4
#define XT_PF4 4
#endif
#ifndef XT_PF3
#define XT_PF3 4
#endif
template <int P, bool REG>
struct Prefetched {  // ... of which this many really are (the rest is read where it is used)
  static constexpr int value = REG ? kPrefetch : (P >= 4 ? XT_PF4 : (P == 3 ? XT_PF3 : kPrefetch));
};

// Which flag sets beyond {none, POST} have specialised multipole handlers in the production build:
// -1: not even the flag-less one, 0: none, 1: PRE+POST, 2: PRE+POST and PRE.  (A case label moved to an impossible key -- order bits that
// cannot occur -- drops its handler from the instantiation.)
#ifndef XT_SET_P4
#define XT_SET_P4 0
#endif
#ifndef XT_SET_P3
#define XT_SET_P3 1
#endif
#ifndef XT_SET_P2
#define XT_SET_P2 1
#endif
template <int P, bool REG>
struct HandlerSet {
  static constexpr int value = P >= 4 ? XT_SET_P4 : (P == 3 ? XT_SET_P3 : XT_SET_P2);
};

// Hot per-thread state of P particles: what drifts and kicks touch at every element.
template <int P>
struct Parts {
  double x[P], px[P], y[P], py[P], zeta[P];
  uint32_t alive;  // bit j: slot j holds a particle that is still being tracked
};

// Cold per-thread state: functions of (delta, ptau), which only a cavity changes.  ptau
// (cavities), delta and rv0v = (1 + beta0 ptau)/(1 + delta) (curved multipoles), opd2 =
// (1 + delta)^2, b = 1 + beta0 ptau and g = ptau (ptau + 2/beta0)/gamma0^2 (drifts).  rpp / rvv are
// written straight to global memory by the cavity map; s / at_turn / at_element / state are
// touched only when a particle is lost and at the end of the launch.
//
// Two homes.  REG = false (large ensembles, 4 CTAs per SM at <= 128 registers): the values live in
// shared memory, one row of 6P doubles per thread at compile-time offsets from one base
// register; the row pitch is odd (in doubles) so that a warp's 64-bit accesses are bank-conflict
// free; the Horner loop keeps the registers for its P independent chains.  REG = true (small
// ensembles that leave the register file half empty, configs[2]: 8 warps per SM): the values stay
// in registers, which takes ~6 LDS and their latency out of every record.
template <int P, bool REG>
struct Cold;

template <int P>
struct Cold<P, false> {
  static constexpr int kPitch = (6 * P) | 1;  // doubles per thread row
  static constexpr bool kInRegs = false;
  double *row;    // this thread's row: P each of ptau, delta, rv0v, opd2, b, g
  int stride;     // blockDim.x
  int64_t first;  // index of slot 0's particle; slot j is first + j * stride
  __device__ __forceinline__ void attach(unsigned char *smem_rows) {
    row = reinterpret_cast<double *>(smem_rows) + static_cast<uint32_t>(kPitch) * threadIdx.x;
  }
  __device__ __forceinline__ double &ptau(int j) { return row[j]; }
  __device__ __forceinline__ double &delta(int j) { return row[P + j]; }
  __device__ __forceinline__ double &rv0v(int j) { return row[2 * P + j]; }
  __device__ __forceinline__ double &opd2(int j) { return row[3 * P + j]; }
  __device__ __forceinline__ double &b(int j) { return row[4 * P + j]; }
  __device__ __forceinline__ double &g(int j) { return row[5 * P + j]; }
  __device__ __forceinline__ int64_t idx(int j) const { return first + static_cast<int64_t>(j) * stride; }
};

template <int P>
struct Cold<P, true> {
  static constexpr int kPitch = 0;  // no shared-memory rows
  static constexpr bool kInRegs = true;
  double v_ptau[P], v_delta[P], v_rv0v[P], v_opd2[P], v_b[P], v_g[P];
  int stride;
  int64_t first;
  __device__ __forceinline__ void attach(unsigned char *) {}
  __device__ __forceinline__ double &ptau(int j) { return v_ptau[j]; }
  __device__ __forceinline__ double &delta(int j) { return v_delta[j]; }
  __device__ __forceinline__ double &rv0v(int j) { return v_rv0v[j]; }
  __device__ __forceinline__ double &opd2(int j) { return v_opd2[j]; }
  __device__ __forceinline__ double &b(int j) { return v_b[j]; }
  __device__ __forceinline__ double &g(int j) { return v_g[j]; }
  __device__ __forceinline__ int64_t idx(int j) const { return first + static_cast<int64_t>(j) * stride; }
};

template <class ColdT>
__device__ __forceinline__ void refresh_cached(ColdT &cold, int j, double opd, double b, double t, double igam2) {
  cold.opd2(j) = opd * opd;
  cold.b(j) = b;
  cold.g(j) = t * igam2;
  cold.rv0v(j) = b / opd;
}

// M2: complex Horner, coefficients stored highest order first as (c[n], s[n]) pairs.
// One step: (re + i im) <- (re + i im)(x + i y) + (c + i s).
template <int P>
__device__ __forceinline__ void horner_step(const double2 c, const double (&x)[P], const double (&y)[P],
                                            double (&re)[P], double (&im)[P]) {
#pragma unroll
  for (int j = 0; j < P; ++j) {
    const double nre = XT_MADD(re[j], x[j], XT_NMADD(im[j], y[j], c.x));  // re*x + (c - im*y)
    const double nim = XT_MADD(re[j], y[j], XT_MADD(im[j], x[j], c.y));   // re*y + (s + im*x)
    re[j] = nre;
    im[j] = nim;
  }
}

// The first step, straight from the leading pair (the same arithmetic as a step from
// re = top.x, im = top.y, without the register copies).
template <int P>
__device__ __forceinline__ void horner_first(const double2 top, const double2 c, const double (&x)[P],
                                             const double (&y)[P], double (&re)[P], double (&im)[P]) {
#pragma unroll
  for (int j = 0; j < P; ++j) {
    re[j] = XT_MADD(top.x, x[j], XT_NMADD(top.y, y[j], c.x));
    im[j] = XT_MADD(top.x, y[j], XT_MADD(top.y, x[j], c.y));
  }
}

// Order known at compile time (the orders a lattice is full of: N = 15 in configs[2-4]): fully unrolled,
// no remainder branches, no loop; every coefficient sits at an immediate offset from the record, so
// the LDS.128 are free to move up.  c0, c1 = the two leading pairs (prefetched before the dispatch).
template <int P, int N>
__device__ __forceinline__ void horner_fixed(const double2 *__restrict__ cs, const double2 c0, const double2 c1,
                                             const double (&x)[P], const double (&y)[P], double (&re)[P],
                                             double (&im)[P]) {
  static_assert(N >= 1, "order 0 has no recurrence");
  horner_first<P>(c0, c1, x, y, re, im);
#pragma unroll
  for (int k = 2; k <= N; ++k) horner_step<P>(cs[k], x, y, re, im);
}

// Any order (run time): (order mod 4) leading steps, then groups of four with the next group's first
// pair loaded one group ahead.
template <int P>
__device__ __forceinline__ void horner(const double2 *__restrict__ cs, int order, const double (&x)[P],
                                       const double (&y)[P], double (&re)[P], double (&im)[P]) {
  const double2 top = cs[0];
  const int rem = order & 3;
  if (rem == 3) {
    horner_first<P>(top, cs[1], x, y, re, im);
    horner_step<P>(cs[2], x, y, re, im);
    horner_step<P>(cs[3], x, y, re, im);
  } else if (rem == 2) {
    horner_first<P>(top, cs[1], x, y, re, im);
    horner_step<P>(cs[2], x, y, re, im);
  } else if (rem == 1) {
    horner_first<P>(top, cs[1], x, y, re, im);
  } else {
#pragma unroll
    for (int j = 0; j < P; ++j) {
      re[j] = top.x;
      im[j] = top.y;
    }
  }
  cs += rem + 1;
  double2 c0 = cs[0];  // first pair of the next group: always one group ahead of its use
#pragma unroll 1
  for (int k = rem + 1; k <= order; k += 4) {
    const double2 c1 = cs[1], c2 = cs[2], c3 = cs[3];
    const double2 n0 = cs[4];  // may lie just past the record (inside the stage buffer's spare bytes): never used then
    cs += 4;
    horner_step<P>(c0, x, y, re, im);
    horner_step<P>(c1, x, y, re, im);
    horner_step<P>(c2, x, y, re, im);
    horner_step<P>(c3, x, y, re, im);
    c0 = n0;
  }
}

// A particle left the aperture: its record is final, so write it now (the thread owns the
// row).  Out of line and by value: the rare path must not force the hot state into memory.
__device__ __noinline__ void store_lost(const xt_particles p, const double *s_table, int64_t i, double x,
                                        double px, double y, double py, double zeta, double delta, double ptau,
                                        uint32_t elem, int64_t turns_done) {
  p.x[i] = x;
  p.px[i] = px;
  p.y[i] = y;
  p.py[i] = py;
  p.zeta[i] = zeta;
  p.delta[i] = delta;
  p.ptau[i] = ptau;
  p.s[i] = s_table[elem];
  p.at_turn[i] += turns_done;
  p.state[i] = 0;
  if (p.at_element) p.at_element[i] = static_cast<int64_t>(elem);
}

// ... and park the slot on the reference orbit, where every map stays finite and cheap.
template <int P, class ColdT>
__device__ __forceinline__ void lose(Parts<P> &q, uint32_t out, ColdT &cold, uint32_t elem, int64_t turns_done,
                                     const TrackArgs &a) {
#pragma unroll
  for (int j = 0; j < P; ++j) {
    if (out & (1u << j)) {
      store_lost(a.p, a.s_table, cold.idx(j), q.x[j], q.px[j], q.y[j], q.py[j], q.zeta[j], cold.delta(j),
                 cold.ptau(j), elem, turns_done);
      q.x[j] = q.px[j] = q.y[j] = q.py[j] = q.zeta[j] = 0.0;
    }
  }
  q.alive &= ~out;
}

// M1 exact drift, cancellation-free zeta (DESIGN.md section 5 "Drift"), in two halves.
// drift_eval computes what depends on (px, py, delta, ptau) only; drift_apply advances
// x, y, zeta by one length.  A drift changes none of the inputs of drift_eval, so
// consecutive drifts share one evaluation: the values are the ones each drift would have
// recomputed, bit for bit.
template <int P>
struct DriftCoef {
  double u[P], v[P], gm[P];  // validation: 1/(pz (pz + b)), pz + b;  production: 1/pz, 1/(pz + b);  g - pxy2
};

template <int P, class ColdT>
__device__ __forceinline__ void drift_eval(const Parts<P> &q, ColdT &cold, DriftCoef<P> &d) {
  double opd2[P], b[P], g[P];
#pragma unroll
  for (int j = 0; j < P; ++j) {
    opd2[j] = cold.opd2(j);
    b[j] = cold.b(j);
    g[j] = cold.g(j);
  }
#pragma unroll
  for (int j = 0; j < P; ++j) {
    const double t1 = XT_MUL(q.px[j], q.px[j]);
    const double pxy2 = XT_MADD(q.py[j], q.py[j], t1);
    const double rad = opd2[j] - pxy2;
#ifdef XT_CANONICAL_DRIFT
    const double pz = sqrt(rad);
    const double s1 = pz + b[j];
    const double den = XT_MUL(pz, s1);
    d.u[j] = 1.0 / den;
    d.v[j] = s1;
#else
    // 1/pz by one cubic Newton step on the RSQ seed; 1/(pz + b) likewise on the RCP seed
    const double r0 = rsqrt_seed(rad);
    const double e = fma(-rad, XT_MUL(r0, r0), 1.0);
    const double r1 = fma(fma(e, 0.375, 0.5), XT_MUL(r0, e), r0);  // 1/pz
    const double s1 = fma(rad, r1, b[j]);                          // pz + b
    const double y0 = rcp_seed(s1);
    const double f = fma(-s1, y0, 1.0);
    d.u[j] = r1;
    d.v[j] = fma(y0, fma(f, f, f), y0);                            // 1/(pz + b)
#endif
    d.gm[j] = g[j] - pxy2;
  }
}

template <int P>
__device__ __forceinline__ void drift_apply(Parts<P> &q, const DriftCoef<P> &d, const double length) {
#pragma unroll
  for (int j = 0; j < P; ++j) {
#ifdef XT_CANONICAL_DRIFT
    const double lr = XT_MUL(length, d.u[j]);   // L/(pz (pz + b))
    const double lpz = XT_MUL(lr, d.v[j]);  // L/pz
#else
    const double lpz = XT_MUL(length, d.u[j]);
    const double lr = XT_MUL(lpz, d.v[j]);
#endif
    q.x[j] = XT_MADD(q.px[j], lpz, q.x[j]);
    q.y[j] = XT_MADD(q.py[j], lpz, q.y[j]);
    q.zeta[j] = XT_MADD(d.gm[j], lr, q.zeta[j]);
  }
}

template <int P, class ColdT>
__device__ __forceinline__ void drift(Parts<P> &q, ColdT &cold, const double length) {
  DriftCoef<P> d;
  drift_eval<P>(q, cold, d);
  drift_apply<P>(q, d, length);
}

// M4: change of reference frame ("tilts, misalignments").
template <int P>
__device__ __forceinline__ void s_rotation(Parts<P> &q, const double2 cs) {  // cs = (cos_z, sin_z)
#pragma unroll
  for (int j = 0; j < P; ++j) {
    const double nx = XT_MADD(cs.x, q.x[j], XT_MUL(cs.y, q.y[j]));
    const double ny = XT_MADD(cs.x, q.y[j], -XT_MUL(cs.y, q.x[j]));
    const double npx = XT_MADD(cs.x, q.px[j], XT_MUL(cs.y, q.py[j]));
    const double npy = XT_MADD(cs.x, q.py[j], -XT_MUL(cs.y, q.px[j]));
    q.x[j] = nx;
    q.y[j] = ny;
    q.px[j] = npx;
    q.py[j] = npy;
  }
}

template <int P>
__device__ __forceinline__ void xy_shift(Parts<P> &q, const double2 d) {  // d = (dx, dy)
#pragma unroll
  for (int j = 0; j < P; ++j) {
    q.x[j] = q.x[j] - d.x;
    q.y[j] = q.y[j] - d.y;
  }
}

// One multipole record: [drift] [shift, rotate] kick [rotate, shift] [drift [drift]] with one
// dispatch.  Slots (xt_internal.h): {l_pre, l_post} {l_post2, wf} [4 misalignment slots] pairs.
// F >= 0 fixes the flag set at compile time (no flag branches), F < 0 reads it from the tag;
// CURVED likewise (1: TAG_CMULT, 0: TAG_MULT, < 0: from the tag); ORDER >= 1 fixes the order (fully
// unrolled Horner, F must not contain TAG_MISAL), ORDER < 0 reads it from the tag.  pf holds the first
// kPrefetch slots of the record, loaded before the dispatch: the two extras and, without
// misalignment, the two leading pairs.
template <int P, int F, int CURVED, int ORDER, class ColdT>
__device__ __forceinline__ void multipole_record(Parts<P> &q, ColdT &cold, const double2 *slots,
                                                 const double2 (&pf)[kPrefetch], const uint32_t tag,
                                                 const double p0) {
  const uint32_t f = F >= 0 ? static_cast<uint32_t>(F) : tag;
  const bool curved = CURVED >= 0 ? (CURVED != 0) : ((tag & TAG_TYPE_MASK) == TAG_CMULT);
  const double2 dl = pf[0];                  // {l_pre, l_post}
  const double2 l2wf = pf[1];                // {l_post2, wf}
  const double2 *mis = slots + 2;            // misalignment slots, if any
  if (f & TAG_PRE) drift<P>(q, cold, dl.x);
  if (f & TAG_MISAL) {
    xy_shift<P>(q, mis[0]);
    s_rotation<P>(q, mis[1]);
  }
  double re[P], im[P];
  if (ORDER >= 1) {
    constexpr int kHave = Prefetched<P, ColdT::kInRegs>::value;
    const double2 *cs = slots + 2;
    horner_fixed<P, (ORDER >= 1 ? ORDER : 1)>(cs, kHave > 2 ? pf[2] : cs[0], kHave > 3 ? pf[3] : cs[1], q.x, q.y, re,
                                               im);
  } else {
    const int order = static_cast<int>((tag >> 8) & 0x7fu);
    horner<P>(slots + ((f & TAG_MISAL) ? 6 : 2), order, q.x, q.y, re, im);
  }
#pragma unroll
  for (int j = 0; j < P; ++j) {
    q.px[j] = q.px[j] - re[j];
    q.py[j] = q.py[j] + im[j];
  }
  if (curved) {
    const double hxl = p0, wf = l2wf.y;
#pragma unroll
    for (int j = 0; j < P; ++j) {
      q.px[j] = XT_MADD(hxl, cold.delta(j), q.px[j]);
      q.px[j] = XT_NMADD(wf, q.x[j], q.px[j]);
      q.zeta[j] = XT_NMADD(XT_MUL(hxl, q.x[j]), cold.rv0v(j), q.zeta[j]);
    }
  }
  if (f & TAG_MISAL) {
    s_rotation<P>(q, mis[2]);
    xy_shift<P>(q, mis[3]);
  }
  if (f & TAG_POST) {
    DriftCoef<P> d;
    drift_eval<P>(q, cold, d);
    drift_apply<P>(q, d, dl.y);
    if (f & TAG_POST2) drift_apply<P>(q, d, l2wf.x);
  }
}

// ---------------------------------------------------------------------------------------------------
// Maps of the extended kernels (thick elements, polygons, radiation, monitors).  They are out of line,
// but take ONE particle by value and return its new coordinates by value: arguments and results travel
// in registers, the callers index their P slots statically, and nothing of the hot state is ever
// forced into local memory (round 1 passed Parts<P>& and indexed it in a rolled loop: 600-2200
// LDL/STL per kernel).
struct Hot {
  double x, px, y, py, zeta;
};
// Inlined into the P-times unrolled callers the thick maps of a thread's P particles interleave (P independent
// chains through sincos / cosh / sinh instead of one); -DXT_THICK_INLINE=__noinline__ keeps one copy out of line.
#ifndef XT_THICK_INLINE
#define XT_THICK_INLINE __forceinline__
#endif

// Thick quadrupole (reading A18): the exact flow of
// H = (px^2 + py^2)/(2(1+delta)) + (k1/2)(x^2 - y^2) over the length.  With w = sqrt(|k1|/(1+delta))
// the focusing plane turns by w L (cos, sin), the other follows cosh, sinh; the path length is
// zeta += L g/((1+delta)((1+delta)+b)) - rv0v/(2(1+delta)^2) int (px^2 + py^2) ds (closed form below).
__device__ XT_THICK_INLINE Hot thick_quadrupole_one(Hot h, const double delta, const double opd2, const double b,
                                                 const double g, const double rv0v, const double k1,
                                                 const double length) {
  const double opd = 1.0 + delta;
  const double rk = k1 / opd;
  const double w = sqrt(fabs(rk));
  const double wl = XT_MUL(w, length);
  double sn, cs;
  sincos(wl, &sn, &cs);
#ifdef XT_FMAD_OFF
  const double ch = cosh(wl), sh = sinh(wl);
  const double h2w = 0.5 / w;
#define XT_OVER_W(a) ((a) / w)
#else
  // production: cosh and sinh from one expm1 (wl >= 0; sinh = (e - 1 + (e - 1)/e)/2 keeps its accuracy for
  // small arguments), and the divisions by w as multiplications by 1/w: ~2 ulp, far inside the 1e-12 bar
  const double em1 = expm1(wl);
  const double ep = em1 + 1.0;
  const double en = 1.0 / ep;
  const double ch = XT_MUL(0.5, ep + en), sh = XT_MUL(0.5, fma(em1, en, em1));
  const double rw = 1.0 / w;
  const double h2w = XT_MUL(0.5, rw);
#define XT_OVER_W(a) XT_MUL((a), rw)
#endif
  const double ow = XT_MUL(opd, w);
  const double iw = 1.0 / ow;
  const bool focus_x = rk > 0.0;
  const double u = focus_x ? h.x : h.y, pu = focus_x ? h.px : h.py;
  const double v = focus_x ? h.y : h.x, pv = focus_x ? h.py : h.px;
  const double au = XT_MUL(ow, u);
  const double av = XT_MUL(ow, v);
  const double u1 = XT_MADD(u, cs, XT_MUL(XT_MUL(pu, iw), sn));
  const double pu1 = XT_NMADD(au, sn, XT_MUL(pu, cs));
  const double v1 = XT_MADD(v, ch, XT_MUL(XT_MUL(pv, iw), sh));
  const double pv1 = XT_MADD(pv, ch, XT_MUL(av, sh));
  const double hl = XT_MUL(0.5, length);
  const double pu2 = XT_MUL(pu, pu), au2 = XT_MUL(au, au), pv2 = XT_MUL(pv, pv), av2 = XT_MUL(av, av);
  const double i_f = XT_MADD(pu2 + au2, hl, XT_MUL(XT_MUL(pu2 - au2, XT_MUL(sn, cs)), h2w)) -
                     XT_OVER_W(XT_MUL(XT_MUL(au, pu), XT_MUL(sn, sn)));
  const double i_d = XT_MADD(pv2 - av2, hl, XT_MUL(XT_MUL(pv2 + av2, XT_MUL(sh, ch)), h2w)) +
                     XT_OVER_W(XT_MUL(XT_MUL(av, pv), XT_MUL(sh, sh)));
#undef XT_OVER_W
  const double slip = XT_MUL(length, g / XT_MUL(opd, opd + b));
  Hot o;
  o.zeta = (h.zeta + slip) - XT_MUL(rv0v / XT_MUL(2.0, opd2), i_f + i_d);
  o.x = focus_x ? u1 : v1;
  o.px = focus_x ? pu1 : pv1;
  o.y = focus_x ? v1 : u1;
  o.py = focus_x ? pv1 : pu1;
  return o;
}

// Thick sector bend, 'expanded' model (reading A19):
// the exact flow of H = (px^2 + py^2)/(2(1+delta)) - h x (1+delta) + k0 x + (k0 h/2) x^2, i.e. the
// thin curved multipole of step M2 smeared over the arc length.  The validation build evaluates the oracle's
// expression tree; the production build multiplies by reciprocals where that tree divides repeatedly.
__device__ XT_THICK_INLINE Hot thick_bend_one(Hot p, const double delta, const double opd2, const double b,
                                           const double g, const double rv, const double k0, const double h,
                                           const double length) {
  const double opd = 1.0 + delta;
  const double w = sqrt(XT_MUL(k0, h) / opd);
  const double wl = XT_MUL(w, length);
  double sn, cs;
  sincos(wl, &sn, &cs);
  const double c1 = 1.0 - cs;
  const double ow = XT_MUL(opd, w);
#ifdef XT_FMAD_OFF
#define XT_OVER_W(a) ((a) / w)
#define XT_OVER_OW(a) ((a) / ow)
  const double h2w = 0.5 / w;
#else
  // production: the nine divisions by w and by (1+delta) w as multiplications by two reciprocals (~2 ulp)
  const double rw = 1.0 / w, row = 1.0 / ow;
#define XT_OVER_W(a) XT_MUL((a), rw)
#define XT_OVER_OW(a) XT_MUL((a), row)
  const double h2w = XT_MUL(0.5, rw);
#endif
  const double fw = XT_OVER_W(XT_NMADD(1.0, k0, XT_MUL(h, opd)));  // (h (1+delta) - k0)/w
  const double x = p.x, px = p.px, py = p.py;
  const double a = XT_MADD(ow, x, -fw);
  const double pw = XT_OVER_OW(px);
  const double x1 = XT_MADD(x, cs, XT_MUL(pw, sn)) + XT_OVER_OW(XT_MUL(fw, c1));
  const double px1 = XT_NMADD(a, sn, XT_MUL(px, cs));
  const double ix = (XT_OVER_W(XT_MUL(x, sn)) + XT_OVER_W(XT_MUL(pw, c1))) + XT_MUL(XT_OVER_OW(fw), length - XT_OVER_W(sn));
  const double px2 = XT_MUL(px, px), a2 = XT_MUL(a, a);
  const double ip = XT_MADD(px2 + a2, XT_MUL(0.5, length), XT_MUL(XT_MUL(px2 - a2, XT_MUL(sn, cs)), h2w)) -
                    XT_OVER_W(XT_MUL(XT_MUL(a, px), XT_MUL(sn, sn)));
#undef XT_OVER_W
#undef XT_OVER_OW
  const double slip = XT_MUL(length, g / XT_MUL(opd, opd + b));
  Hot o;
  o.zeta = ((p.zeta + slip) - XT_MUL(XT_MUL(rv, h), ix)) -
           XT_MUL(rv / XT_MUL(2.0, opd2), ip + XT_MUL(length, XT_MUL(py, py)));
  o.y = XT_MUL(length, py) / opd + p.y;
  o.py = py;
  o.x = x1;
  o.px = px1;
  return o;
}

// Thick sector bend, 'full' model ("a 'full' map, which is appropriate for small accelerators";
// DESIGN.md reading A23): the helix of a charge in the uniform field k0, cut by the exit plane of the frame
// of curvature h, in the cancellation-free form of the oracle (same arithmetic order).
__device__ XT_THICK_INLINE Hot thick_bend_full_one(Hot p, const double delta, const double opd2, const double b,
                                                   const double ptau, const double beta0, const double k0,
                                                   const double h, const double length) {
  const double x = p.x, px = p.px, py = p.py;
  const double t1 = XT_MUL(px, px);
  const double pxy2 = XT_MADD(py, py, t1);
  const double pz = sqrt(opd2 - pxy2);
  const double dpz = XT_NMADD(1.0, pxy2, XT_MUL(delta, delta + 2.0)) / (pz + 1.0);  // pz - 1
  const double eps = (k0 - h) / h;
  const double cc = XT_NMADD(k0, x, dpz - eps);
  const double th = XT_MUL(h, length);
  const double sn = sin(th);
  const double sh = sin(XT_MUL(0.5, th));
  const double c1 = XT_MUL(2.0, XT_MUL(sh, sh));  // 1 - cos
  const double dpx = XT_NMADD(px, c1, XT_MUL(cc, sn));
  const double px1 = px + dpx;
  const double ph2 = XT_NMADD(py, py, opd2);
  const double pz1 = sqrt(XT_NMADD(px1, px1, ph2));
  const double num = XT_MADD(px, sn, XT_MUL(c1, cc)) - XT_MUL(dpx, px + px1) / (pz1 + pz);
  const double iph = 1.0 / sqrt(ph2);
  const double dd = asin(XT_MUL(px, iph)) - asin(XT_MUL(px1, iph));
  Hot o;
  o.x = num / k0 + x;
  o.y = XT_MUL(py, th + dd) / k0 + p.y;
  o.zeta = (p.zeta + XT_MUL(XT_NMADD(h, XT_MUL(beta0, ptau), k0 - h), length) / k0) - XT_MUL(b, dd) / k0;
  o.px = px1;
  o.py = py;
  return o;
}

template <int P, class ColdT>
__device__ __forceinline__ void thick_bend_full(Parts<P> &q, ColdT &cold, const double k0, const double h,
                                                const double length, const double beta0) {
#pragma unroll
  for (int j = 0; j < P; ++j) {
    const Hot o = thick_bend_full_one(Hot{q.x[j], q.px[j], q.y[j], q.py[j], q.zeta[j]}, cold.delta(j), cold.opd2(j),
                                      cold.b(j), cold.ptau(j), beta0, k0, h, length);
    q.x[j] = o.x;
    q.px[j] = o.px;
    q.y[j] = o.y;
    q.py[j] = o.py;
    q.zeta[j] = o.zeta;
  }
}

template <int P, class ColdT>
__device__ __forceinline__ void thick_quadrupole(Parts<P> &q, ColdT &cold, const double k1, const double length) {
#pragma unroll
  for (int j = 0; j < P; ++j) {
    const Hot o = thick_quadrupole_one(Hot{q.x[j], q.px[j], q.y[j], q.py[j], q.zeta[j]}, cold.delta(j), cold.opd2(j),
                                       cold.b(j), cold.g(j), cold.rv0v(j), k1, length);
    q.x[j] = o.x;
    q.px[j] = o.px;
    q.y[j] = o.y;
    q.py[j] = o.py;
    q.zeta[j] = o.zeta;
  }
}

template <int P, class ColdT>
__device__ __forceinline__ void thick_bend(Parts<P> &q, ColdT &cold, const double k0, const double h,
                                           const double length) {
#pragma unroll
  for (int j = 0; j < P; ++j) {
    const Hot o = thick_bend_one(Hot{q.x[j], q.px[j], q.y[j], q.py[j], q.zeta[j]}, cold.delta(j), cold.opd2(j),
                                 cold.b(j), cold.g(j), cold.rv0v(j), k0, h, length);
    q.x[j] = o.x;
    q.px[j] = o.px;
    q.y[j] = o.y;
    q.py[j] = o.py;
    q.zeta[j] = o.zeta;
  }
}

// A: elliptical aperture (x^2 b^2 + y^2 a^2 <= a^2 b^2, edge inclusive, NaN lost).
template <int P, class ColdT>
__device__ __forceinline__ void limit_ellipse(Parts<P> &q, ColdT &cold, const double2 ba, const double a2b2,
                                              uint32_t elem, int64_t turns_done, const TrackArgs &a) {
  uint32_t out = 0;
#pragma unroll
  for (int j = 0; j < P; ++j) {
    const double tt = XT_MADD(XT_MUL(q.x[j], q.x[j]), ba.x, XT_MUL(XT_MUL(q.y[j], q.y[j]), ba.y));
    out |= (tt <= a2b2) ? 0u : (1u << j);
  }
  out &= q.alive;
  if (out) lose<P>(q, out, cold, elem, turns_done, a);
}

// A: polygon aperture (even-odd rule; reading A20): the half line from the particle towards +x
// crosses edge (v[i-1] -> v[i]) iff its ends lie on different sides of the horizontal through the particle
// and the crossing point is to the right of it.  NaN crosses nothing: lost.  THICK kernels only.
template <int P, class ColdT>
__device__ __forceinline__ void limit_polygon(Parts<P> &q, ColdT &cold, const double2 *v, int n, uint32_t elem,
                                              int64_t turns_done, const TrackArgs &a) {
  uint32_t in = 0;
  double2 vj = v[n - 1];
#pragma unroll 1
  for (int i = 0; i < n; ++i) {
    const double2 vi = v[i];
#pragma unroll
    for (int j = 0; j < P; ++j) {
      const double y = q.y[j];
      if ((vi.y > y) != (vj.y > y)) {
        const double xc = XT_MUL(vj.x - vi.x, y - vi.y) / (vj.y - vi.y) + vi.x;
        if (q.x[j] < xc) in ^= (1u << j);
      }
    }
    vj = vi;
  }
  const uint32_t out = ~in & q.alive;
  if (out) lose<P>(q, out, cold, elem, turns_done, a);
}

// Thin multipole with "mean" synchrotron radiation (reading A22, section 18): the
// fraction r = krad (1+delta) kick^2 / lpath of the particle's energy is radiated, half before the kick and
// half after; delta follows from the energy as behind a cavity, px and py shrink with the momentum.
// slots: (c[n], s[n]) pairs n = N .. 0 with c[0] = knl[0] - hxl, {wf, length}, {krad, 0}.  THICK kernels only.
// One particle by value in, its new state by value out (see Hot above).
struct RadOut {
  double px, py, zeta, ptau, delta, opd, b, t;
};

__device__ __noinline__ RadOut rad_multipole_one(const double x, const double y, double px, double py, double zeta,
                                                 double ptau, double delta, const double2 *slots, const int order,
                                                 const double hxl, const double beta0, const double tib) {
  const double2 wl = slots[order + 1], kr = slots[order + 2];
  const double ib = 1.0 / beta0;
  double re = slots[0].x, im = slots[0].y;
#pragma unroll 1
  for (int n = 1; n <= order; ++n) {
    const double2 c = slots[n];
    const double nre = XT_MADD(re, x, XT_NMADD(im, y, c.x));
    const double nim = XT_MADD(re, y, XT_MADD(im, x, c.y));
    re = nre;
    im = nim;
  }
  const double dpxf = XT_NMADD(wl.x, x, -re - hxl);  // the field's kick (re has the curvature folded in)
  const double dpyf = im;
  const double kick2 = XT_MADD(dpxf, dpxf, XT_MUL(dpyf, dpyf));
  const double lpath = XT_MADD(hxl, x, wl.y);
  RadOut o{};
#pragma unroll 1
  for (int half = 0; half < 2; ++half) {
    const double opd = 1.0 + delta;
    const double rh = XT_MUL(0.5 * kr.x, XT_MUL(opd, kick2)) / lpath;
    ptau = XT_NMADD(rh, ptau + ib, ptau);
    const double t = XT_MUL(ptau, ptau + tib);
    delta = t / (sqrt(t + 1.0) + 1.0);
    const double opd1 = 1.0 + delta;
    const double f = opd1 / opd;
    px = XT_MUL(px, f);
    py = XT_MUL(py, f);
    const double b = XT_MADD(beta0, ptau, 1.0);
    o.opd = opd1;
    o.b = b;
    o.t = t;
    if (half == 0) {  // the thin kick itself, in the arithmetic of the plain multipole
      px = px - re;
      py = py + im;
      px = XT_MADD(hxl, delta, px);
      px = XT_NMADD(wl.x, x, px);
      zeta = XT_NMADD(XT_MUL(hxl, x), b / opd1, zeta);  // b/opd1 = the refreshed rv0v
    }
  }
  o.px = px;
  o.py = py;
  o.zeta = zeta;
  o.ptau = ptau;
  o.delta = delta;
  return o;
}

template <int P, class ColdT>
__device__ __forceinline__ void rad_multipole(Parts<P> &q, ColdT &cold, const double2 *slots, int order, double hxl,
                                              const TrackArgs &a) {
#pragma unroll
  for (int j = 0; j < P; ++j) {
    if (!(q.alive & (1u << j))) continue;
    const RadOut o = rad_multipole_one(q.x[j], q.y[j], q.px[j], q.py[j], q.zeta[j], cold.ptau(j), cold.delta(j), slots,
                                       order, hxl, a.beta0, a.tib);
    q.px[j] = o.px;
    q.py[j] = o.py;
    q.zeta[j] = o.zeta;
    cold.ptau(j) = o.ptau;
    cold.delta(j) = o.delta;
    refresh_cached(cold, j, o.opd, o.b, o.t, a.igam2);
    a.p.rpp[cold.idx(j)] = 1.0 / o.opd;
    a.p.rvv[cold.idx(j)] = o.opd / o.b;
  }
}

// Internal monitor record (xt_twiss4d_line): row p0 of the monitor buffer (TrackArgs::monitor_rows, set per
// call: no process-global state) receives the coordinates of every alive particle of this thread.
// THICK kernels only.
template <int P, class ColdT>
__device__ __forceinline__ void monitor_store(const Parts<P> &q, ColdT &cold, double row, const TrackArgs &a) {
  double *base = a.monitor_rows + static_cast<int64_t>(row) * a.n_part * 6;
#pragma unroll
  for (int j = 0; j < P; ++j) {
    if (q.alive & (1u << j)) {
      double *o = base + cold.idx(j) * 6;
      o[0] = q.x[j];
      o[1] = q.px[j];
      o[2] = q.y[j];
      o[3] = q.py[j];
      o[4] = q.zeta[j];
      o[5] = cold.delta(j);
    }
  }
}

// Push the P particles of this thread through every record of one staged chunk.
// Returns the position just behind the chunk (where the next chunk of the image starts).
//
// Dispatch: a switch on type | flags [| order] of the (warp-uniform) tag.  The records a thin
// drift-kick-drift lattice is made of -- multipoles (straight and curved) with the flag sets none, POST,
// POST+POST2, PRE+POST+POST2 -- have handlers in which flags and curvature are compile-time constants.
// Lattices whose multipoles are mostly of one order (the packer counts: order 15 in configs[2-4]) run the
// NFIX instantiation, where that order is a compile-time constant too: no remainder branches, a fully
// unrolled Horner whose coefficient loads all sit at immediate offsets.  Every other multipole takes the
// same code with flags and order read at run time.
template <int P, bool THICK, int NFIX, class ColdT>
__device__ __forceinline__ const unsigned char *track_chunk(Parts<P> &q, const unsigned char *rp, ColdT &cold,
                                                            int64_t turns_done, const TrackArgs &a) {
  uint32_t tag = reinterpret_cast<const RecHdr *>(rp)->next;  // chunk preamble
  rp += sizeof(RecHdr);
  while ((tag & TAG_TYPE_MASK) != TAG_END) {
    const RecHdr h = *reinterpret_cast<const RecHdr *>(rp);  // {tag of the NEXT record, elem, p0}
    const double2 *slots = reinterpret_cast<const double2 *>(rp + sizeof(RecHdr));
    // the first slots, loaded before the dispatch resolves (whatever the record is; at the end
    // of a chunk this reads up to 64 spare bytes behind it)
    constexpr int kHave = Prefetched<P, ColdT::kInRegs>::value;
    const double2 zero2 = make_double2(0.0, 0.0);
    const double2 pf[kPrefetch] = {slots[0], slots[1], kHave > 2 ? slots[2] : zero2, kHave > 3 ? slots[3] : zero2};
    const double p0 = h.p0;
    const uint32_t elem = h.elem;
    rp += tag >> 16;  // record size in bytes
    // NFIX > 0: the multipole order(s) with fully unrolled handlers, first | second << 5 (the switch key then
    // includes the order); NFIX = 0: the flag sets are specialised, the order is read at run time.
    constexpr uint32_t kKeyMask = NFIX > 0 ? 0x7fffu : 0xffu;  // type | flags [| order << 8]
    constexpr uint32_t kOrd = NFIX > 0 ? static_cast<uint32_t>(NFIX & 31) : 0u;
    constexpr int kOrdT = NFIX > 0 ? (NFIX & 31) : -1;
    constexpr uint32_t kOrdB = static_cast<uint32_t>(NFIX >> 5);          // second fixed order, 0: none
    constexpr int kOrdBT = (NFIX >> 5) > 0 ? (NFIX >> 5) : 1;
    constexpr uint32_t kNoB = (NFIX >> 5) > 0 ? 0u : 0x6000u;             // parks the second order's labels
    const uint32_t key = tag & kKeyMask;
    switch (key) {
      case TAG_DRIFT:
      case TAG_DRIFT | TAG_POST: {
        DriftCoef<P> d;
        drift_eval<P>(q, cold, d);
        drift_apply<P>(q, d, p0);
        if (tag & TAG_POST) drift_apply<P>(q, d, pf[0].x);  // a second drift, same (px, py)
        break;
      }
#define XT_MULT_CASE(F, N, NT)                                                 \
  case TAG_MULT | (F) | ((N) << 8):                                            \
    multipole_record<P, (F), 0, (NT)>(q, cold, slots, pf, tag, p0);            \
    break;                                                                     \
  case TAG_CMULT | (F) | ((N) << 8):                                           \
    multipole_record<P, (F), 1, (NT)>(q, cold, slots, pf, tag, p0);            \
    break;
      // The flag sets a drift-kick-drift lattice produces.  In the validation build every drift arrives on its
      // own (POST2 records); in the production build consecutive drifts arrive merged, and which of the
      // remaining sets get a specialised handler is a per-shape choice measured on configs[2] / [3]
      // (profiles/r02_shape_sweep.md): every extra handler lengthens the dispatch and the code.
#ifdef XT_FMAD_OFF
      XT_MULT_CASE(0u, kOrd, kOrdT)
#else
      XT_MULT_CASE((HandlerSet<P, ColdT::kInRegs>::value >= 0 ? 0u : 0x7000u), kOrd, kOrdT)
#endif
      XT_MULT_CASE(TAG_POST, kOrd, kOrdT)
      XT_MULT_CASE(kNoB, kOrdB, kOrdBT)  // the second fixed order (lattices of thin quadrupoles and sextupoles)
      XT_MULT_CASE(TAG_POST | kNoB, kOrdB, kOrdBT)
#ifdef XT_FMAD_OFF
      XT_MULT_CASE(TAG_POST | TAG_POST2, kOrd, kOrdT)
      XT_MULT_CASE(TAG_PRE | TAG_POST | TAG_POST2, kOrd, kOrdT)
#else
      XT_MULT_CASE(TAG_PRE | TAG_POST | (HandlerSet<P, ColdT::kInRegs>::value >= 1 ? 0u : 0x7000u), kOrd, kOrdT)
      XT_MULT_CASE(TAG_PRE | (HandlerSet<P, ColdT::kInRegs>::value >= 2 ? 0u : 0x7000u), kOrd, kOrdT)
#endif
#undef XT_MULT_CASE
      case TAG_CAVITY: {
        const double2 kv = pf[0];  // (kz, vn)
#pragma unroll
        for (int j = 0; j < P; ++j) {
          if (q.alive & (1u << j)) {
            const double phase = XT_NMADD(kv.x, q.zeta[j], p0);
            const double ptau = XT_MADD(kv.y, sin(phase), cold.ptau(j));
            const double t = XT_MUL(ptau, ptau + a.tib);
            const double delta = t / (sqrt(t + 1.0) + 1.0);
            const double opd = 1.0 + delta;
            const double b = XT_MADD(a.beta0, ptau, 1.0);
            cold.ptau(j) = ptau;
            cold.delta(j) = delta;
            a.p.rpp[cold.idx(j)] = 1.0 / opd;
            a.p.rvv[cold.idx(j)] = opd / b;
            refresh_cached(cold, j, opd, b, t, a.igam2);
          }
        }
        break;
      }
      case TAG_SROT:
      case TAG_SROT | TAG_POST: {
        s_rotation<P>(q, pf[0]);
        if (tag & TAG_POST) xy_shift<P>(q, pf[1]);  // rotation, then shift: the way out of a misaligned magnet
        break;
      }
      case TAG_SHIFT:
      case TAG_SHIFT | TAG_POST: {
        xy_shift<P>(q, pf[0]);
        if (tag & TAG_POST) s_rotation<P>(q, pf[1]);  // shift, then rotation: the way in
        break;
      }
      case TAG_RECT: {
        const double2 xr = pf[0], yr = pf[1];
        uint32_t out = 0;
#pragma unroll
        for (int j = 0; j < P; ++j) {
          const bool inside = (q.x[j] >= xr.x) && (q.x[j] <= xr.y) && (q.y[j] >= yr.x) && (q.y[j] <= yr.y);
          out |= inside ? 0u : (1u << j);
        }
        out &= q.alive;
        if (out) lose<P>(q, out, cold, elem, turns_done, a);
        break;
      }
      case TAG_ELLIPSE: {
        limit_ellipse<P>(q, cold, pf[0], p0, elem, turns_done, a);  // pf[0] = (b2, a2), p0 = a2 b2
        break;
      }
      default: {
        const uint32_t type = tag & TAG_TYPE_MASK;
        if (type == TAG_MULT || type == TAG_CMULT) {
          // any other order or flag set (misaligned magnets): everything read at run time
          multipole_record<P, -1, -1, -1>(q, cold, slots, pf, tag, p0);
        } else if (THICK) {  // the extended maps: only lattices that contain them run these instantiations
          const int order = static_cast<int>((tag >> 8) & 0x7fu);
          if (type == TAG_QUAD) thick_quadrupole<P>(q, cold, p0, pf[0].x);                 // p0 = k1, {length, 0}
          else if (type == TAG_BEND) thick_bend<P>(q, cold, p0, pf[0].x, pf[0].y);         // p0 = k0, {h, length}
          else if (type == TAG_BENDF) thick_bend_full<P>(q, cold, p0, pf[0].x, pf[0].y, a.beta0);
          else if (type == TAG_RMULT) rad_multipole<P>(q, cold, slots, order, p0, a);      // p0 = hxl
          else if (type == TAG_MON) monitor_store<P>(q, cold, p0, a);                      // p0 = row
          else if (type == TAG_POLY)  // (record bytes - header) / 16 vertices
            limit_polygon<P>(q, cold, slots, static_cast<int>(((tag >> 16) - sizeof(RecHdr)) / 16), elem, turns_done, a);
        }
        break;
      }
    }
    if (tag & TAG_APER) {
      // the record ends with an elliptical aperture: {b2, a2}, {a2 b2, element index} are its last slots
      const double2 ba = *reinterpret_cast<const double2 *>(rp - 32);
      const double2 ce = *reinterpret_cast<const double2 *>(rp - 16);
      limit_ellipse<P>(q, cold, ba, ce.x, static_cast<uint32_t>(ce.y), turns_done, a);
    }
    tag = h.next;
  }
  return rp;
}

// Register budget per thread (CTAs of 128 threads: 65536 / (128 * CTAs per SM)).
#ifndef XT_REGS3
#define XT_REGS3 128
#endif
#ifndef XT_REGS4
#define XT_REGS4 128
#endif
#ifndef XT_REGS3R
#define XT_REGS3R 255
#endif
// (CTAs are at most 256 threads: xt_api.cu)
// The extended kernels call the out-of-line thick maps: their small shapes get room for the call's live
// state (at 64 / 80 registers they spilled ~100 values around every call).
template <int P, bool REG, bool THICK>
struct RegBudget {
  static constexpr int value = REG ? (P == 4 ? 168 : (P == 3 ? XT_REGS3R : (P == 2 ? 168 : 96)))
                                   : (P == 1 ? (THICK ? 96 : 64) : (P == 2 ? (THICK ? 128 : 80) : (P == 3 ? XT_REGS3 : XT_REGS4)));
};

// Shared memory: [0,16) two mbarriers; [128, 128 + 8*kPitch*blockDim) cold per-thread rows (none when
// the cold state lives in registers); then staging buffer 0 (and buffer 1 for multi-chunk lattices),
// 128-byte aligned, and 64 spare bytes (the record prefetch and the run-time Horner loop read up to four
// slots past the record they are in; the values are never used).
template <int P, bool THICK, bool REG, int NFIX>
__global__ void __maxnreg__((RegBudget<P, REG, THICK>::value)) xt_track_kernel(const TrackArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  const uint32_t bar0 = smem_addr(smem);
  using ColdT = Cold<P, REG>;
  ColdT cold;
  cold.attach(smem + 128);
  cold.stride = static_cast<int>(blockDim.x);
  unsigned char *const buf0 =
      smem + 128 + ((static_cast<uint32_t>(8 * ColdT::kPitch) * blockDim.x + 127u) & ~127u);

  if constexpr (!REG) {
    // The shapes with the cold state in shared memory: one share of the ensemble per CTA for the whole launch.
    // Balanced hand-out (device side, so that compaction's device counter needs no host
    // sync): use as few CTAs as hold n_active particles, rounded up to a whole number per SM,
    // and give each the same share.
    const int64_t n_active = a.n_active ? *a.n_active : a.n_part;
    const int64_t cap = static_cast<int64_t>(blockDim.x) * P;
    const int64_t need = (n_active + cap - 1) / cap;
    int64_t used = ((need + a.grid_quantum - 1) / a.grid_quantum) * a.grid_quantum;
    if (used > static_cast<int64_t>(gridDim.x)) used = gridDim.x;
    if (static_cast<int64_t>(blockIdx.x) >= used) return;  // CTA-uniform
    const int64_t share = (n_active + used - 1) / used;
    const int64_t start = static_cast<int64_t>(blockIdx.x) * share;
    if (start >= n_active) return;  // CTA-uniform
    const int64_t count = (n_active - start < share) ? n_active - start : share;

    Parts<P> q;
    cold.first = start + threadIdx.x;
    q.alive = 0;
#pragma unroll
    for (int j = 0; j < P; ++j) {
      const int64_t k = static_cast<int64_t>(j) * blockDim.x + threadIdx.x;
      const int64_t i = start + k;
      const bool live = (k < count) && (a.p.state[i] == 1);
      if (live) {
        q.x[j] = a.p.x[i];
        q.px[j] = a.p.px[i];
        q.y[j] = a.p.y[i];
        q.py[j] = a.p.py[i];
        q.zeta[j] = a.p.zeta[i];
        const double delta = a.p.delta[i];
        const double ptau = a.p.ptau[i];
        cold.delta(j) = delta;
        cold.ptau(j) = ptau;
        q.alive |= 1u << j;
        const double opd = 1.0 + delta;
        const double b = XT_MADD(a.beta0, ptau, 1.0);
        const double t = XT_MUL(ptau, ptau + a.tib);
        refresh_cached(cold, j, opd, b, t, a.igam2);
      } else {
        q.x[j] = q.px[j] = q.y[j] = q.py[j] = q.zeta[j] = 0.0;
        cold.opd2(j) = cold.b(j) = 1.0;
        cold.g(j) = 0.0;
        cold.ptau(j) = cold.delta(j) = 0.0;
        cold.rv0v(j) = 1.0;
      }
    }

    const bool single = (a.n_chunks == 1);
    if (threadIdx.x == 0) {
      mbar_init(bar0, 1);
      mbar_init(bar0 + 8, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // A stage = stage_chunks consecutive chunks = one bulk copy into one buffer.  A lattice that fits one
    // chunk is loaded once and stays resident in buffer 0: its warps run free, no CTA-level
    // synchronisation; otherwise the stages alternate between the two buffers and a __syncthreads_or at
    // the end of each releases the buffer and tells the CTA whether anyone is still alive.  One loop (and
    // one copy of the record interpreter in the instruction cache) serves both.
    const int32_t m = a.stage_chunks;
    const int32_t n_stages = (a.n_chunks + m - 1) / m;
    const uint32_t stage_bytes = static_cast<uint32_t>(m) * a.chunk_bytes;
    auto load_stage = [&](int32_t sidx, uint32_t nb) {  // thread 0 only
      const int32_t first = sidx * m;
      const int32_t last = (first + m < a.n_chunks ? first + m : a.n_chunks) - 1;
      const ChunkDesc d0 = a.chunks[first], d1 = a.chunks[last];
      const uint32_t bytes = static_cast<uint32_t>(d1.offset + d1.nbytes - d0.offset);
      tma_load_chunk(bar0 + 8 * nb, smem_addr(buf0 + static_cast<size_t>(nb) * stage_bytes), a.image + d0.offset,
                     bytes);
    };
    if (threadIdx.x == 0) load_stage(0, 0);
    if (single) mbar_wait(bar0, 0);
    const int64_t total = a.n_turns * n_stages;
    int64_t turns_done = 0;
    int64_t gidx = 0;  // global stage counter: buffer = gidx & 1, phase parity = (gidx >> 1) & 1
    int32_t c = 0;
    bool any = true;
    while (gidx < total) {
      uint32_t cb = 0;
      if (!single) {
        if (threadIdx.x == 0 && gidx + 1 < total) {
          // buffer (gidx+1)&1 was released by the __syncthreads_or that ended iteration gidx-1
          load_stage((c + 1 == n_stages) ? 0 : c + 1, static_cast<uint32_t>((gidx + 1) & 1));
        }
        cb = static_cast<uint32_t>(gidx & 1);
        mbar_wait(bar0 + 8 * cb, static_cast<uint32_t>((gidx >> 1) & 1));
      }
      const bool warp_alive = __any_sync(0xffffffffu, q.alive != 0);
      if (single && !warp_alive) break;  // this warp is done; the others do not wait for it
      if (warp_alive) {
        const int32_t n_sub = (c * m + m < a.n_chunks ? m : a.n_chunks - c * m);
        const unsigned char *rp = buf0 + static_cast<size_t>(cb) * stage_bytes;
        for (int32_t k = 0; k < n_sub; ++k) rp = track_chunk<P, THICK, NFIX>(q, rp, cold, turns_done, a);
      }
      ++gidx;
      if (++c == n_stages) {
        c = 0;
        ++turns_done;  // T: turn completed
      }
      if (!single) {
        any = __syncthreads_or(q.alive != 0 ? 1 : 0) != 0;
        if (!any) break;
      }
    }
    if (!single && !any && gidx < total) {
      // every particle of the CTA is lost: drain the copy still in flight before exiting
      mbar_wait(bar0 + 8 * static_cast<uint32_t>(gidx & 1), static_cast<uint32_t>((gidx >> 1) & 1));
    }

    // W: survivors (lost particles were written when they were lost; rpp, rvv by the cavities)
#pragma unroll
    for (int j = 0; j < P; ++j) {
      if (q.alive & (1u << j)) {
        const int64_t i = cold.idx(j);
        a.p.x[i] = q.x[j];
        a.p.px[i] = q.px[j];
        a.p.y[i] = q.y[j];
        a.p.py[i] = q.py[j];
        a.p.zeta[i] = q.zeta[j];
        a.p.delta[i] = cold.delta(j);
        a.p.ptau[i] = cold.ptau(j);
        a.p.s[i] = 0.0;
        a.p.at_turn[i] += turns_done;
      }
    }
  } else {
    // The small-ensemble shapes (cold state in registers): the same, or the balanced mode.
    // Balanced mode (compiled into the shapes that keep the cold state in registers: the one-wave
    // ensembles).  An ensemble of G groups on S resident CTAs, G / S not an integer, leaves lanes or whole
    // CTA slots empty for the whole run when every CTA owns its particles (configs[2]: 5.28 warp-slots per
    // scheduler run as 6).  Here the work is cut into items (group g of blockDim.x * P particles, block k of
    // a few turns) and the launch has one CTA per item; the hardware starts a CTA whenever a slot is free.
    // A first-in first-out queue in device memory holds the groups that are ready for their next block:
    // the first G pop tickets are block 0 of each group; a CTA that has stored block k of a group pushes
    // the group's next item, and pop ticket G + n takes push number n (spinning until it is there).  A
    // group in the queue is taken by the next CTA that starts, so no group waits while an SM has room, and
    // an SM on which a CTA waits runs its other CTAs faster: the load evens out over the run.  Tickets are
    // taken in the order the CTAs start and every push is made by a running CTA, so nothing can deadlock.
    // The state of a group goes through HBM between its blocks.
    // queue[0]: pop tickets, queue[1]: pushes, queue[2]: groups that are through, queue[4 + n]: item of push n,
  // plus one (0: not there yet).
    const bool queued = a.queue != nullptr;
    __shared__ unsigned int s_item;
    int64_t start, count, n_turns, t0 = 0;
    unsigned int item = 0, n_groups = 0;
    if (queued) {
      // with compaction the number of particles (and of groups) is a device counter; the launch then has
      // CTAs for the largest number of items there can be, and the ones left over leave when every group
      // has done its last block (queue[2])
      const int64_t cap = static_cast<int64_t>(blockDim.x) * P;
      const int64_t n_act = a.n_active ? *a.n_active : a.n_part;
      n_groups = static_cast<unsigned int>((n_act + cap - 1) / cap);
      if (threadIdx.x == 0) {
        const unsigned int my = atomicAdd(a.queue, 1u);
        unsigned int it = my;
        if (my >= n_groups) {
          const unsigned int *slot = a.queue + 4 + (my - n_groups);
          it = 0xffffffffu;
          for (unsigned int spin = 0;; ++spin) {
            unsigned int v, fin;
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(slot) : "memory");
            if (v != 0u) {
              it = v - 1u;
              break;
            }
            if ((spin & 7u) == 7u) {  // now and then: is everything through?
              asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(fin) : "l"(a.queue + 2) : "memory");
              if (fin >= n_groups) {  // nothing will be pushed any more (a push precedes the count it enables)
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(slot) : "memory");
                if (v != 0u) it = v - 1u;
                break;
              }
            }
            __nanosleep(1000);  // an item lasts milliseconds
          }
          __threadfence();
        }
        s_item = it;
      }
      __syncthreads();
      item = s_item;
      if (item == 0xffffffffu) return;  // CTA-uniform: a CTA left over
      const unsigned int grp = item % n_groups;
      const unsigned int blk = item / n_groups;
      start = static_cast<int64_t>(grp) * cap;
      count = (n_act - start < cap) ? n_act - start : cap;
      const int64_t l0 = first_block_turns(grp, a.block_turns);
      t0 = blk == 0 ? 0 : l0 + static_cast<int64_t>(blk - 1) * a.block_turns;
      const int64_t len = blk == 0 ? l0 : static_cast<int64_t>(a.block_turns);
      n_turns = (a.n_turns - t0 < len) ? a.n_turns - t0 : len;
    } else {
      // Balanced hand-out (device side, so that compaction's device counter needs no host
      // sync): use as few CTAs as hold n_active particles, rounded up to a whole number per SM,
      // and give each the same share.
      const int64_t n_active = a.n_active ? *a.n_active : a.n_part;
      const int64_t cap = static_cast<int64_t>(blockDim.x) * P;
      const int64_t need = (n_active + cap - 1) / cap;
      int64_t used = ((need + a.grid_quantum - 1) / a.grid_quantum) * a.grid_quantum;
      if (used > static_cast<int64_t>(gridDim.x)) used = gridDim.x;
      if (static_cast<int64_t>(blockIdx.x) >= used) return;  // CTA-uniform
      const int64_t share = (n_active + used - 1) / used;
      start = static_cast<int64_t>(blockIdx.x) * share;
      if (start >= n_active) return;  // CTA-uniform
      count = (n_active - start < share) ? n_active - start : share;
      n_turns = a.n_turns;
    }

    Parts<P> q;
    cold.first = start + threadIdx.x;
    q.alive = 0;
#pragma unroll
    for (int j = 0; j < P; ++j) {
      const int64_t k = static_cast<int64_t>(j) * blockDim.x + threadIdx.x;
      const int64_t i = start + k;
      const bool live = (k < count) && (__ldcg(a.p.state + i) == 1);
      if (live) {
        q.x[j] = __ldcg(a.p.x + i);
        q.px[j] = __ldcg(a.p.px + i);
        q.y[j] = __ldcg(a.p.y + i);
        q.py[j] = __ldcg(a.p.py + i);
        q.zeta[j] = __ldcg(a.p.zeta + i);
        const double delta = __ldcg(a.p.delta + i);
        const double ptau = __ldcg(a.p.ptau + i);
        cold.delta(j) = delta;
        cold.ptau(j) = ptau;
        q.alive |= 1u << j;
        const double opd = 1.0 + delta;
        const double b = XT_MADD(a.beta0, ptau, 1.0);
        const double t = XT_MUL(ptau, ptau + a.tib);
        refresh_cached(cold, j, opd, b, t, a.igam2);
      } else {
        q.x[j] = q.px[j] = q.y[j] = q.py[j] = q.zeta[j] = 0.0;
        cold.opd2(j) = cold.b(j) = 1.0;
        cold.g(j) = 0.0;
        cold.ptau(j) = cold.delta(j) = 0.0;
        cold.rv0v(j) = 1.0;
      }
    }

    const bool single = (a.n_chunks == 1);
    if (threadIdx.x == 0) {
      mbar_init(bar0, 1);
      mbar_init(bar0 + 8, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // A stage = stage_chunks consecutive chunks = one bulk copy into one buffer.  A lattice that fits one
    // chunk is loaded once and stays resident in buffer 0: its warps run free, no CTA-level
    // synchronisation; otherwise the stages alternate between the two buffers and a __syncthreads_or at
    // the end of each releases the buffer and tells the CTA whether anyone is still alive.  One loop (and
    // one copy of the record interpreter in the instruction cache) serves both.
    const int32_t m = a.stage_chunks;
    const int32_t n_stages = (a.n_chunks + m - 1) / m;
    const uint32_t stage_bytes = static_cast<uint32_t>(m) * a.chunk_bytes;
    auto load_stage = [&](int32_t sidx, uint32_t nb) {  // thread 0 only
      const int32_t first = sidx * m;
      const int32_t last = (first + m < a.n_chunks ? first + m : a.n_chunks) - 1;
      const ChunkDesc d0 = a.chunks[first], d1 = a.chunks[last];
      const uint32_t bytes = static_cast<uint32_t>(d1.offset + d1.nbytes - d0.offset);
      tma_load_chunk(bar0 + 8 * nb, smem_addr(buf0 + static_cast<size_t>(nb) * stage_bytes), a.image + d0.offset,
                     bytes);
    };
    if (threadIdx.x == 0) load_stage(0, 0);
    if (single) mbar_wait(bar0, 0);
    const int64_t total = n_turns * n_stages;
    int64_t turns_done = 0;
    int64_t gidx = 0;  // global stage counter: buffer = gidx & 1, phase parity = (gidx >> 1) & 1
    int32_t c = 0;
    bool any = true;
    while (gidx < total) {
      uint32_t cb = 0;
      if (!single) {
        if (threadIdx.x == 0 && gidx + 1 < total) {
          // buffer (gidx+1)&1 was released by the __syncthreads_or that ended iteration gidx-1
          load_stage((c + 1 == n_stages) ? 0 : c + 1, static_cast<uint32_t>((gidx + 1) & 1));
        }
        cb = static_cast<uint32_t>(gidx & 1);
        mbar_wait(bar0 + 8 * cb, static_cast<uint32_t>((gidx >> 1) & 1));
      }
      const bool warp_alive = __any_sync(0xffffffffu, q.alive != 0);
      if (single && !warp_alive) break;  // this warp is done; the others do not wait for it
      if (warp_alive) {
        const int32_t n_sub = (c * m + m < a.n_chunks ? m : a.n_chunks - c * m);
        const unsigned char *rp = buf0 + static_cast<size_t>(cb) * stage_bytes;
        for (int32_t k = 0; k < n_sub; ++k) rp = track_chunk<P, THICK, NFIX>(q, rp, cold, turns_done, a);
      }
      ++gidx;
      if (++c == n_stages) {
        c = 0;
        ++turns_done;  // T: turn completed
      }
      if (!single) {
        any = __syncthreads_or(q.alive != 0 ? 1 : 0) != 0;
        if (!any) break;
      }
    }
    if (!single && !any && gidx < total) {
      // every particle of the CTA is lost: drain the copy still in flight before exiting
      mbar_wait(bar0 + 8 * static_cast<uint32_t>(gidx & 1), static_cast<uint32_t>((gidx >> 1) & 1));
    }

    // W: survivors (lost particles were written when they were lost; rpp, rvv by the cavities)
#pragma unroll
    for (int j = 0; j < P; ++j) {
      if (q.alive & (1u << j)) {
        const int64_t i = cold.idx(j);
        a.p.x[i] = q.x[j];
        a.p.px[i] = q.px[j];
        a.p.y[i] = q.y[j];
        a.p.py[i] = q.py[j];
        a.p.zeta[i] = q.zeta[j];
        a.p.delta[i] = cold.delta(j);
        a.p.ptau[i] = cold.ptau(j);
        a.p.s[i] = 0.0;
        a.p.at_turn[i] = __ldcg(a.p.at_turn + i) + turns_done;
      }
    }
    if (queued) {
      // publish: every thread's stores, then the group's next item (release), or one group fewer to wait for
      __syncthreads();
      if (threadIdx.x == 0) {
        __threadfence();
        if (t0 + n_turns < a.n_turns) {
          const unsigned int n = atomicAdd(a.queue + 1, 1u);
          const unsigned int next = item + n_groups + 1u;
          asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(a.queue + 4 + n), "r"(next) : "memory");
        } else {
          atomicAdd(a.queue + 2, 1u);
        }
      }
    }
  }
}

__global__ void xt_init_derived_kernel(xt_particles p, int64_t n, double beta0, double ib, double ib2) {
  const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= n) return;
  // DESIGN.md section 5 "Init helper": ptau = t/(sqrt(t + 1/beta0^2) + 1/beta0), t = delta(delta+2)
  const double d = p.delta[i];
  const double t = d * (d + 2.0);
  const double pt = t / (sqrt(t + ib2) + ib);
  const double opd = 1.0 + d;
  const double b = 1.0 + beta0 * pt;
  p.ptau[i] = pt;
  p.rpp[i] = 1.0 / opd;
  p.rvv[i] = opd / b;
}

// Per device and instantiation, once: opt in to large dynamic shared memory, prefer shared memory over
// L1 (every hot read is a shared-memory broadcast) and read the register count the occupancy rule below
// needs.  (Round 1 made these three driver calls on every launch; xt_track_knobs launches once per turn.)
constexpr int kMaxDevices = 64;
template <int P, bool THICK, bool REG, int NFIX>
int kernel_registers(int device, int *regs) {
  static std::atomic<int> cache[kMaxDevices];  // 0: not configured yet
  const int slot = (device >= 0 && device < kMaxDevices) ? device : -1;
  if (slot >= 0) {
    const int v = cache[slot].load(std::memory_order_acquire);
    if (v > 0) {
      *regs = v;
      return XT_OK;
    }
  }
  XT_CUDA(cudaFuncSetAttribute(xt_track_kernel<P, THICK, REG, NFIX>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  XT_CUDA(cudaFuncSetAttribute(xt_track_kernel<P, THICK, REG, NFIX>, cudaFuncAttributePreferredSharedMemoryCarveout,
                               cudaSharedmemCarveoutMaxShared));
  cudaFuncAttributes fa;
  XT_CUDA(cudaFuncGetAttributes(&fa, xt_track_kernel<P, THICK, REG, NFIX>));
  *regs = fa.numRegs > 0 ? fa.numRegs : 128;
  if (slot >= 0) cache[slot].store(*regs, std::memory_order_release);
  return XT_OK;
}

// Items of the balanced mode: about this many lattice records each (configs[2]: 4 turns, 9 ms), at most
// kMaxBlocks blocks of turns per launch (the queue has one word per item), at least six, and more groups
// than SMs (else every CTA has an SM of its own).
constexpr int64_t kItemRecords = 12000;
constexpr int64_t kMaxBlocks = 256;
constexpr int64_t kMinBlocks = 6;

template <int P, bool THICK, bool REG, int NFIX>
int launch_track_pt(const TrackArgs &a, const xt_lattice *lat, int block, int balance, cudaStream_t st) {
  const size_t cold_bytes =
      (static_cast<size_t>(8 * Cold<P, REG>::kPitch) * block + 127) & ~static_cast<size_t>(127);
  const int64_t cap = static_cast<int64_t>(block) * P;
  const int64_t need = (a.n_part + cap - 1) / cap;
  int64_t grid = ((need + a.grid_quantum - 1) / a.grid_quantum) * a.grid_quantum;
  if (grid > 2147483647LL) {
    set_error("xt_track: too many particles for one launch");
    return XT_ERR_INVALID_ARG;
  }
  int regs = 128;
  const int rc = kernel_registers<P, THICK, REG, NFIX>(lat->device, &regs);
  if (rc != XT_OK) return rc;
  const int64_t by_regs = 65536 / (static_cast<int64_t>(regs) * block) > 0 ? 65536 / (static_cast<int64_t>(regs) * block) : 1;
  TrackArgs b = a;
  if (!REG) b.queue = nullptr;
  if (b.queue) {
    const int64_t t = balance_block_turns(lat, a.n_turns, balance);
    const int64_t n_blocks = (a.n_turns + t - 1) / t;
    const bool worth = balance > 0 || (n_blocks >= kMinBlocks && need > a.grid_quantum);
    if (worth && need * (n_blocks + 1) < 2000000000LL && t < 2000000000LL && need < 4000000) {
      b.block_turns = static_cast<int32_t>(t);
      // one CTA per item, the hardware starts them as slots become free: a first item of 1 .. t turns per
      // group, then blocks of t turns (an upper bound: the CTAs left over leave when every group is through)
      grid = need * (1 + (a.n_turns - 1 + t - 1) / t);
    } else {
      b.queue = nullptr;
    }
  }
  // Staging depth: as many chunks per bulk copy (fewer CTA-wide barriers per turn) as shared memory
  // allows without taking a resident CTA away.
  // (In the balanced mode no more CTAs of an SM run at a time than there are groups per SM: configs[2] has
  // 2.64, three resident CTAs with four chunks per stage do better than four with two, 0.612 against 0.603.)
  int64_t resident = by_regs;
  const int64_t per_sm = ((b.queue ? need : grid) + a.grid_quantum - 1) / a.grid_quantum;
  if (resident > per_sm) resident = per_sm;
  if (resident < 1) resident = 1;
  b.stage_chunks = 1;
  const size_t chunk = static_cast<size_t>(lat->info.chunk_bytes);
  auto smem_for = [&](int m) { return 128 + 64 + cold_bytes + (lat->info.n_chunks == 1 ? 1 : 2) * m * chunk; };
  for (int m = 4; m > 1; m >>= 1) {
    if (lat->info.n_chunks >= 2 * m && smem_for(m) <= 96 * 1024 &&
        static_cast<size_t>(resident) * (smem_for(m) + 1024) <= 227 * 1024) {
      b.stage_chunks = m;
      break;
    }
  }
  const size_t smem = smem_for(b.stage_chunks);
  xt_track_kernel<P, THICK, REG, NFIX><<<static_cast<unsigned>(grid), block, smem, st>>>(b);
  count_launch();
  XT_CUDA(cudaGetLastError());
  return XT_OK;
}

// Lattices with thick elements take the instantiation that has their maps compiled in; lattices full of
// order-15 multipoles the one with the unrolled order-15 handlers (3 and 4 particles per thread: the
// shapes large lattices run with).
constexpr int kFixedOrder = 15;       // configs[2-4]: every magnet carries errors up to order 15
constexpr int kFixedLow = 1 | (2 << 5);  // thin quadrupoles and sextupoles (configs[0], [1]): orders 1 and 2
template <int P, bool REG>
int launch_track_p(const TrackArgs &a, const xt_lattice *lat, int block, int balance, cudaStream_t st) {
  constexpr bool kHasFixed = (P >= 3) || REG;  // which shapes exist with the unrolled order-15 handlers
  if (kHasFixed && lat->fixed_order == kFixedOrder) {
    constexpr int NF = kHasFixed ? kFixedOrder : 0;
    return lat->extended ? launch_track_pt<P, true, REG, NF>(a, lat, block, balance, st)
                         : launch_track_pt<P, false, REG, NF>(a, lat, block, balance, st);
  }
  if (!REG && lat->fixed_order == kFixedLow) {
    constexpr int NF = REG ? 0 : kFixedLow;
    return lat->extended ? launch_track_pt<P, true, REG, NF>(a, lat, block, balance, st)
                         : launch_track_pt<P, false, REG, NF>(a, lat, block, balance, st);
  }
  return lat->extended ? launch_track_pt<P, true, REG, 0>(a, lat, block, balance, st)
                       : launch_track_pt<P, false, REG, 0>(a, lat, block, balance, st);
}

}  // namespace

// ppt: particles per thread (1, 2, 3, 4); cold_in_regs: the cold per-particle state in registers
// instead of shared memory (instantiated for 3 particles per thread: the small-ensemble shape).
int64_t balance_block_turns(const xt_lattice *lat, int64_t n_turns, int balance) {
  const int64_t rec = lat->info.n_records > 0 ? lat->info.n_records : 1;
  int64_t t = balance > 1 ? balance : (kItemRecords + rec - 1) / rec;
  if (t < (n_turns + kMaxBlocks - 1) / kMaxBlocks) t = (n_turns + kMaxBlocks - 1) / kMaxBlocks;
  if (t > n_turns) t = n_turns;
  return t > 0 ? t : 1;
}

bool balance_pays(const xt_lattice *lat, int64_t n_turns, int balance) {
  if (balance < 0 || n_turns <= 0) return false;
  if (balance > 0) return true;
  // the shapes with the cold state in registers have no handlers with the orders 1 and 2 fixed
  if (lat->fixed_order == kFixedLow) return false;
  const int64_t t = balance_block_turns(lat, n_turns, balance);
  return (n_turns + t - 1) / t >= kMinBlocks;
}

size_t balance_scratch_bytes(int64_t n_part, int block, int ppt) {
  const int64_t cap = static_cast<int64_t>(block) * ppt;
  const int64_t need = cap > 0 ? (n_part + cap - 1) / cap : 0;
  return (static_cast<size_t>(need * kMaxBlocks + 4) * sizeof(unsigned int) + 255) & ~static_cast<size_t>(255);
}

int launch_track(const xt_lattice *lat, const xt_particles &p, int64_t n_part, const int64_t *d_n_active,
                 int64_t n_turns, int block, int ppt, bool cold_in_regs, cudaStream_t st, unsigned int *queue,
                 int balance) {
  if (n_part <= 0 || n_turns <= 0) return XT_OK;
  TrackArgs a;
  a.image = lat->d_image;
  a.chunks = lat->d_chunks;
  a.s_table = lat->d_s_table;
  a.n_active = d_n_active;
  a.monitor_rows = lat->d_monitor_rows;
  a.p = p;
  a.n_part = n_part;
  a.n_turns = n_turns;
  a.n_chunks = static_cast<int32_t>(lat->info.n_chunks);
  a.chunk_bytes = static_cast<uint32_t>(lat->info.chunk_bytes);
  a.grid_quantum = lat->n_sm > 0 ? lat->n_sm : 1;
  a.beta0 = lat->k.beta0;
  a.tib = lat->k.tib;
  a.igam2 = lat->k.igam2;
  a.queue = (cold_in_regs && balance >= 0) ? queue : nullptr;
  a.block_turns = 0;
  if (a.queue) {  // tickets and per-group counters start from zero
    XT_CUDA(cudaMemsetAsync(a.queue, 0, balance_scratch_bytes(n_part, block, ppt), st));
  }
  if (cold_in_regs) {
    if (ppt == 1) return launch_track_p<1, true>(a, lat, block, balance, st);
    if (ppt == 2) return launch_track_p<2, true>(a, lat, block, balance, st);
    if (ppt == 3) return launch_track_p<3, true>(a, lat, block, balance, st);
    if (ppt == 4) return launch_track_p<4, true>(a, lat, block, balance, st);
    set_error("xt_track: particles_per_thread must be 1, 2, 3 or 4");
    return XT_ERR_INVALID_ARG;
  }
  switch (ppt) {
    case 1:
      return launch_track_p<1, false>(a, lat, block, balance, st);
    case 2:
      return launch_track_p<2, false>(a, lat, block, balance, st);
    case 3:
      return launch_track_p<3, false>(a, lat, block, balance, st);
    case 4:
      return launch_track_p<4, false>(a, lat, block, balance, st);
    default:
      set_error("xt_track: particles_per_thread must be 1, 2, 3 or 4");
      return XT_ERR_INVALID_ARG;
  }
}

int launch_init_derived(const xt_lattice *lat, const xt_particles &p, int64_t n, cudaStream_t st) {
  if (n <= 0) return XT_OK;
  const int block = 256;
  const int64_t grid = (n + block - 1) / block;
  xt_init_derived_kernel<<<static_cast<unsigned>(grid), block, 0, st>>>(p, n, lat->k.beta0, lat->k.ib, lat->k.ib2);
  count_launch();
  XT_CUDA(cudaGetLastError());
  return XT_OK;
}

}  // namespace xt
