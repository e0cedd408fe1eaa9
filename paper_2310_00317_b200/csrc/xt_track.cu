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
// share (warp-uniform); a record is usually a fused [drift] kick [drift drift] group
// (xt_internal.h).  Multipoles are a complex Horner recurrence of FMAs.
//
// Why P > 1 (profiles/r01b_track_p1_summary.md): with one particle per thread 58 % of the
// issued warp instructions were not FP64 (dispatch, LDS, branches, the slow-path guards of
// sqrt and /) and the FP64 pipe sat at 49 %.  P particles per thread share every one of those
// instructions and give each warp P independent FP64 chains.
//
// Arithmetic.  The maps are written in the canonical order of DESIGN.md section 5 through
// XT_MADD / XT_NMADD / XT_MUL.  The validation build (--fmad=false, XT_FMAD_OFF) evaluates
// exactly those trees with IEEE sqrt and division and is bit-identical to the oracle on
// cavity-free lattices.  The production build fuses every a*b + c into one DFMA (explicitly,
// so that results do not depend on the launch shape) and replaces the drift's sqrt + division
// by branch-free Newton sequences on the MUFU.RSQ64H / MUFU.RCP64H seeds (DESIGN.md section
// 6.3): same formula, <= 2 ulp on the increments; the measured distance to the oracle is set by
// FMA fusion, not by this block (<= 0.5 of the 1e-12 bar either way).
#include "xt_internal.h"

namespace xt {
namespace {

struct TrackArgs {
  const unsigned char *image;
  const ChunkDesc *chunks;
  const double *s_table;
  const int64_t *n_active;  // device counter (compaction path) or nullptr
  xt_particles p;
  int64_t n_part;
  int64_t n_turns;
  int32_t n_chunks;
  uint32_t chunk_bytes;
  int32_t stage_chunks;  // consecutive chunks staged by one bulk copy (they are contiguous in the image)
  int32_t grid_quantum;  // CTAs are handed out in multiples of this (the SM count)
  double beta0, tib, igam2;
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

// Where the thick quadrupole sits in the dispatch.  Its record never occurs in a thin lattice, but
// the presence of the case label reshapes the compare tree ptxas builds for the switch: measured,
// the 3-particle kernel is 1.2 % faster with the label (configs[2]) and the 4-particle one 1 %
// faster without it (configs[3]).  So the thin 4-particle kernel parks the label on a key that
// cannot occur (the switch key is 8 bits wide, the compiler drops the case).
template <int P, bool THICK>
struct QuadCase {
  static constexpr uint32_t value = (P == 4 && !THICK) ? 0x1ffu : static_cast<uint32_t>(TAG_QUAD);
};

template <bool THICK>
struct BendCase {  // thin kernels keep the dispatch tree they were measured with: the label is parked there
  static constexpr uint32_t value = THICK ? static_cast<uint32_t>(TAG_BEND) : 0x2ffu;
};

template <bool THICK>
struct RadCase {
  static constexpr uint32_t value = THICK ? static_cast<uint32_t>(TAG_RMULT) : 0x5ffu;
};

template <bool THICK>
struct MonCase {
  static constexpr uint32_t value = THICK ? static_cast<uint32_t>(TAG_MON) : 0x4ffu;
};

template <bool THICK>
struct PolyCase {
  static constexpr uint32_t value = THICK ? static_cast<uint32_t>(TAG_POLY) : 0x3ffu;
};

constexpr int kPrefetch = 4;  // 16-byte slots of a record loaded ahead of its dispatch ...
#ifndef XT_PF4
#define XT_PF4 2
#endif
#ifndef XT_PF3
#define XT_PF3 2
#endif
template <int P>
struct Prefetched {  // ... of which this many really are (the rest is read where it is used)
  static constexpr int value = P >= 4 ? XT_PF4 : (P == 3 ? XT_PF3 : kPrefetch);
};

// Hot per-thread state of P particles: what drifts and kicks touch at every element.
template <int P>
struct Parts {
  double x[P], px[P], y[P], py[P], zeta[P];
  uint32_t alive;  // bit j: slot j holds a particle that is still being tracked
};

// Cold per-thread state, kept out of the register file (the Horner loop needs the
// registers to interleave its P independent chains): functions of (delta, ptau), which only
// a cavity changes.  ptau (cavities), delta and rv0v = (1 + beta0 ptau)/(1 + delta) (curved
// multipoles), opd2 = (1 + delta)^2, b = 1 + beta0 ptau and g = ptau (ptau + 2/beta0)/gamma0^2
// (drifts) live in shared memory, one row of 6P doubles per thread at compile-time offsets
// from one base register; the row pitch is odd (in doubles) so that a warp's 64-bit
// accesses are bank-conflict free.  rpp / rvv are written straight to global memory by the
// cavity map; s / at_turn / at_element / state are touched only when a particle is lost and
// at the end of the launch.
template <int P>
struct Cold {
  static constexpr int kPitch = (6 * P) | 1;  // doubles per thread row
  double *row;    // this thread's row: P each of ptau, delta, rv0v, opd2, b, g
  int stride;     // blockDim.x
  int64_t first;  // index of slot 0's particle; slot j is first + j * stride
  __device__ __forceinline__ double &ptau(int j) const { return row[j]; }
  __device__ __forceinline__ double &delta(int j) const { return row[P + j]; }
  __device__ __forceinline__ double &rv0v(int j) const { return row[2 * P + j]; }
  __device__ __forceinline__ double &opd2(int j) const { return row[3 * P + j]; }
  __device__ __forceinline__ double &b(int j) const { return row[4 * P + j]; }
  __device__ __forceinline__ double &g(int j) const { return row[5 * P + j]; }
  __device__ __forceinline__ int64_t idx(int j) const { return first + static_cast<int64_t>(j) * stride; }
};

template <int P>
__device__ __forceinline__ void refresh_cached(const Cold<P> &cold, int j, double opd, double b, double t,
                                               double igam2) {
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

// pf = the first kPrefetch pairs, already in registers; the rest comes from cs (shared memory).
template <int P>
__device__ __forceinline__ void horner(const double2 *__restrict__ cs, const double2 (&pf)[kPrefetch], int order,
                                       const double (&x)[P], const double (&y)[P], double (&re)[P],
                                       double (&im)[P]) {
  static_assert(kPrefetch == 4, "the leading steps below take exactly the four leading pairs");
  constexpr int kHave = Prefetched<P>::value;
  // (order mod 4) leading steps, then groups of four
  const double2 top = pf[0];
  const int rem = order & 3;
  if (rem == 3) {
    const double2 c2 = kHave > 2 ? pf[2] : cs[2], c3 = kHave > 3 ? pf[3] : cs[3];
    horner_first<P>(top, pf[1], x, y, re, im);
    horner_step<P>(c2, x, y, re, im);
    horner_step<P>(c3, x, y, re, im);
  } else if (rem == 2) {
    const double2 c2 = kHave > 2 ? pf[2] : cs[2];
    horner_first<P>(top, pf[1], x, y, re, im);
    horner_step<P>(c2, x, y, re, im);
  } else if (rem == 1) {
    horner_first<P>(top, pf[1], x, y, re, im);
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
    const double2 n0 = cs[4];  // may lie just past the record: never used then
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
template <int P>
__device__ __forceinline__ void lose(Parts<P> &q, uint32_t out, const Cold<P> &cold, uint32_t elem,
                                     int64_t turns_done, const TrackArgs &a) {
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

template <int P>
__device__ __forceinline__ void drift_eval(const Parts<P> &q, const Cold<P> &cold, DriftCoef<P> &d) {
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

template <int P>
__device__ __forceinline__ void drift(Parts<P> &q, const Cold<P> &cold, const double length) {
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
// dispatch.  F >= 0 fixes the flag set at compile time (no flag branches), F < 0 reads it
// from the tag; CURVED likewise (1: TAG_CMULT, 0: TAG_MULT, < 0: from the tag).  pf holds the
// first kPrefetch slots of the record, loaded before the dispatch.
template <int P, int F, int CURVED>
__device__ __forceinline__ void multipole_record(Parts<P> &q, const Cold<P> &cold, const double2 *slots,
                                                 const double2 (&pf)[kPrefetch], const uint32_t tag,
                                                 const double p0) {
  const uint32_t f = F >= 0 ? static_cast<uint32_t>(F) : tag;
  const bool curved = CURVED >= 0 ? (CURVED != 0) : ((tag & TAG_TYPE_MASK) == TAG_CMULT);
  const int order = static_cast<int>((tag >> 8) & 0x7fu);
  const double2 *extra = slots + order + 1;  // behind the coefficient pairs
  double wf = 0.0;
  double2 dl = make_double2(0.0, 0.0);
  double l_post2 = 0.0;
  if (curved) wf = (extra++)->x;
  if (f & (TAG_PRE | TAG_POST)) dl = *extra++;
  if (f & TAG_POST2) l_post2 = (extra++)->x;
  if (f & TAG_PRE) drift<P>(q, cold, dl.x);
  if (f & TAG_MISAL) {
    xy_shift<P>(q, extra[0]);
    s_rotation<P>(q, extra[1]);
  }
  double re[P], im[P];
  horner<P>(slots, pf, order, q.x, q.y, re, im);
#pragma unroll
  for (int j = 0; j < P; ++j) {
    q.px[j] = q.px[j] - re[j];
    q.py[j] = q.py[j] + im[j];
  }
  if (curved) {
    const double hxl = p0;
#pragma unroll
    for (int j = 0; j < P; ++j) {
      q.px[j] = XT_MADD(hxl, cold.delta(j), q.px[j]);
      q.px[j] = XT_NMADD(wf, q.x[j], q.px[j]);
      q.zeta[j] = XT_NMADD(XT_MUL(hxl, q.x[j]), cold.rv0v(j), q.zeta[j]);
    }
  }
  if (f & TAG_MISAL) {
    s_rotation<P>(q, extra[2]);
    xy_shift<P>(q, extra[3]);
  }
  if (f & TAG_POST) {
    DriftCoef<P> d;
    drift_eval<P>(q, cold, d);
    drift_apply<P>(q, d, dl.y);
    if (f & TAG_POST2) drift_apply<P>(q, d, l_post2);
  }
}

// Thick quadrupole (reading A18): the exact flow of
// H = (px^2 + py^2)/(2(1+delta)) + (k1/2)(x^2 - y^2) over the length.  With w = sqrt(|k1|/(1+delta))
// the focusing plane turns by w L (cos, sin), the other follows cosh, sinh; the path length is
// zeta += L g/((1+delta)((1+delta)+b)) - rv0v/(2(1+delta)^2) int (px^2 + py^2) ds (closed form below).
// The sign of k1/(1+delta) is the sign of k1 for every physical particle: a warp-uniform branch.
// Only compiled into the THICK instantiations of the kernel: lattices without thick elements run
// the same code as before.
template <int P>
__device__ __noinline__ void thick_quadrupole(Parts<P> &q, const Cold<P> &cold, const double k1, const double length) {
#pragma unroll 1
  for (int j = 0; j < P; ++j) {
    const double opd = 1.0 + cold.delta(j);
    const double rk = k1 / opd;
    const double w = sqrt(fabs(rk));
    const double wl = XT_MUL(w, length);
    double sn, cs;
    sincos(wl, &sn, &cs);
    const double ch = cosh(wl), sh = sinh(wl);
    const double ow = XT_MUL(opd, w);
    const double iw = 1.0 / ow;
    const bool focus_x = rk > 0.0;
    const double u = focus_x ? q.x[j] : q.y[j], pu = focus_x ? q.px[j] : q.py[j];
    const double v = focus_x ? q.y[j] : q.x[j], pv = focus_x ? q.py[j] : q.px[j];
    const double au = XT_MUL(ow, u);
    const double av = XT_MUL(ow, v);
    const double u1 = XT_MADD(u, cs, XT_MUL(XT_MUL(pu, iw), sn));
    const double pu1 = XT_NMADD(au, sn, XT_MUL(pu, cs));
    const double v1 = XT_MADD(v, ch, XT_MUL(XT_MUL(pv, iw), sh));
    const double pv1 = XT_MADD(pv, ch, XT_MUL(av, sh));
    const double hl = XT_MUL(0.5, length);
    const double h2w = 0.5 / w;
    const double pu2 = XT_MUL(pu, pu), au2 = XT_MUL(au, au), pv2 = XT_MUL(pv, pv), av2 = XT_MUL(av, av);
    const double i_f = XT_MADD(pu2 + au2, hl, XT_MUL(XT_MUL(pu2 - au2, XT_MUL(sn, cs)), h2w)) -
                       XT_MUL(XT_MUL(au, pu), XT_MUL(sn, sn)) / w;
    const double i_d = XT_MADD(pv2 - av2, hl, XT_MUL(XT_MUL(pv2 + av2, XT_MUL(sh, ch)), h2w)) +
                       XT_MUL(XT_MUL(av, pv), XT_MUL(sh, sh)) / w;
    const double slip = XT_MUL(length, cold.g(j) / XT_MUL(opd, opd + cold.b(j)));
    q.zeta[j] = (q.zeta[j] + slip) - XT_MUL(cold.rv0v(j) / XT_MUL(2.0, cold.opd2(j)), i_f + i_d);
    if (focus_x) {
      q.x[j] = u1;
      q.px[j] = pu1;
      q.y[j] = v1;
      q.py[j] = pv1;
    } else {
      q.y[j] = u1;
      q.py[j] = pu1;
      q.x[j] = v1;
      q.px[j] = pv1;
    }
  }
}

// Thick sector bend, 'expanded' model (reading A19):
// the exact flow of H = (px^2 + py^2)/(2(1+delta)) - h x (1+delta) + k0 x + (k0 h/2) x^2, i.e. the
// thin curved multipole of step M2 smeared over the arc length.  Same arithmetic as the oracle's.
template <int P>
__device__ __noinline__ void thick_bend(Parts<P> &q, const Cold<P> &cold, const double k0, const double h,
                                        const double length) {
#pragma unroll 1
  for (int j = 0; j < P; ++j) {
    const double opd = 1.0 + cold.delta(j);
    const double w = sqrt(XT_MUL(k0, h) / opd);
    const double wl = XT_MUL(w, length);
    double sn, cs;
    sincos(wl, &sn, &cs);
    const double c1 = 1.0 - cs;
    const double ow = XT_MUL(opd, w);
    const double fw = XT_NMADD(1.0, k0, XT_MUL(h, opd)) / w;  // (h (1+delta) - k0)/w
    const double x = q.x[j], px = q.px[j], py = q.py[j];
    const double a = XT_MADD(ow, x, -fw);
    const double pw = px / ow;
    const double x1 = XT_MADD(x, cs, XT_MUL(pw, sn)) + XT_MUL(fw, c1) / ow;
    const double px1 = XT_NMADD(a, sn, XT_MUL(px, cs));
    const double ix = (XT_MUL(x, sn) / w + XT_MUL(pw, c1) / w) + XT_MUL(fw / ow, length - sn / w);
    const double px2 = XT_MUL(px, px), a2 = XT_MUL(a, a);
    const double ip = XT_MADD(px2 + a2, XT_MUL(0.5, length), XT_MUL(XT_MUL(px2 - a2, XT_MUL(sn, cs)), 0.5 / w)) -
                      XT_MUL(XT_MUL(a, px), XT_MUL(sn, sn)) / w;
    const double rv = cold.rv0v(j);
    const double slip = XT_MUL(length, cold.g(j) / XT_MUL(opd, opd + cold.b(j)));
    q.zeta[j] = ((q.zeta[j] + slip) - XT_MUL(XT_MUL(rv, h), ix)) -
                XT_MUL(rv / XT_MUL(2.0, cold.opd2(j)), ip + XT_MUL(length, XT_MUL(py, py)));
    q.y[j] = XT_MUL(length, py) / opd + q.y[j];
    q.x[j] = x1;
    q.px[j] = px1;
  }
}

// A: elliptical aperture (x^2 b^2 + y^2 a^2 <= a^2 b^2, edge inclusive, NaN lost).
template <int P>
__device__ __forceinline__ void limit_ellipse(Parts<P> &q, const Cold<P> &cold, const double2 ba, const double a2b2,
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
template <int P>
__device__ __noinline__ void limit_polygon(Parts<P> &q, const Cold<P> &cold, const double2 *v, int n, uint32_t elem,
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
template <int P>
__device__ __noinline__ void rad_multipole(Parts<P> &q, const Cold<P> &cold, const double2 *slots, int order,
                                           double hxl, const TrackArgs &a) {
  const double2 wl = slots[order + 1], kr = slots[order + 2];
  const double ib = 1.0 / a.beta0;
#pragma unroll
  for (int j = 0; j < P; ++j) {
    if (!(q.alive & (1u << j))) continue;
    const double x = q.x[j], y = q.y[j];
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
    double px = q.px[j], py = q.py[j], ptau = cold.ptau(j), delta = cold.delta(j);
#pragma unroll 1
    for (int half = 0; half < 2; ++half) {
      const double opd = 1.0 + delta;
      const double rh = XT_MUL(0.5 * kr.x, XT_MUL(opd, kick2)) / lpath;
      ptau = XT_NMADD(rh, ptau + ib, ptau);
      const double t = XT_MUL(ptau, ptau + a.tib);
      delta = t / (sqrt(t + 1.0) + 1.0);
      const double opd1 = 1.0 + delta;
      const double f = opd1 / opd;
      px = XT_MUL(px, f);
      py = XT_MUL(py, f);
      const double b = XT_MADD(a.beta0, ptau, 1.0);
      refresh_cached<P>(cold, j, opd1, b, t, a.igam2);
      if (half == 0) {  // the thin kick itself, in the arithmetic of the plain multipole
        px = px - re;
        py = py + im;
        px = XT_MADD(hxl, delta, px);
        px = XT_NMADD(wl.x, x, px);
        q.zeta[j] = XT_NMADD(XT_MUL(hxl, x), cold.rv0v(j), q.zeta[j]);
      } else {
        a.p.rpp[cold.idx(j)] = 1.0 / opd1;
        a.p.rvv[cold.idx(j)] = opd1 / b;
      }
    }
    q.px[j] = px;
    q.py[j] = py;
    cold.ptau(j) = ptau;
    cold.delta(j) = delta;
  }
}

// Internal monitor record (xt_twiss4d_line): row p0 of the monitor buffer receives the coordinates of every
// alive particle of this thread.  THICK kernels only.
__constant__ double *g_monitor_rows;

template <int P>
__device__ __noinline__ void monitor_store(const Parts<P> &q, const Cold<P> &cold, double row, int64_t n_part) {
  double *base = g_monitor_rows + static_cast<int64_t>(row) * n_part * 6;
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
template <int P, bool THICK>
__device__ __forceinline__ const unsigned char *track_chunk(Parts<P> &q, const unsigned char *rp,
                                                            const Cold<P> &cold, int64_t turns_done,
                                                            const TrackArgs &a) {
  uint32_t tag = reinterpret_cast<const RecHdr *>(rp)->next;  // chunk preamble
  rp += sizeof(RecHdr);
  while ((tag & TAG_TYPE_MASK) != TAG_END) {
    const RecHdr h = *reinterpret_cast<const RecHdr *>(rp);  // {tag of the NEXT record, elem, p0}
    const double2 *slots = reinterpret_cast<const double2 *>(rp + sizeof(RecHdr));
    // the first slots, loaded before the dispatch resolves (whatever the record is; at the end
    // of a chunk this reads up to 64 spare bytes behind it)
    constexpr int kHave = Prefetched<P>::value;
    const double2 zero2 = make_double2(0.0, 0.0);
    const double2 pf[kPrefetch] = {slots[0], slots[1], kHave > 2 ? slots[2] : zero2, kHave > 3 ? slots[3] : zero2};
    const double p0 = h.p0;
    const uint32_t elem = h.elem;
    rp += tag >> 16;  // record size in bytes
    switch (tag & 0xffu) {  // type | flags
      case TAG_DRIFT:
      case TAG_DRIFT | TAG_POST: {
        DriftCoef<P> d;
        drift_eval<P>(q, cold, d);
        drift_apply<P>(q, d, p0);
        if (tag & TAG_POST) drift_apply<P>(q, d, pf[0].x);  // a second drift, same (px, py)
        break;
      }
#define XT_MULT_CASE(F)                                                        \
  case TAG_MULT | (F):                                                         \
    multipole_record<P, (F), 0>(q, cold, slots, pf, tag, p0);                  \
    break;                                                                     \
  case TAG_CMULT | (F):                                                        \
    multipole_record<P, (F), 1>(q, cold, slots, pf, tag, p0);                  \
    break;
      // the flag sets a drift-kick-drift lattice is made of, specialised at compile time ...
      XT_MULT_CASE(0)
      XT_MULT_CASE(TAG_POST)
      XT_MULT_CASE(TAG_POST | TAG_POST2)
      XT_MULT_CASE(TAG_PRE | TAG_POST | TAG_POST2)
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
            refresh_cached<P>(cold, j, opd, b, t, a.igam2);
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
      case QuadCase<P, THICK>::value: {  // thick quadrupole (see QuadCase)
        if (THICK) thick_quadrupole<P>(q, cold, p0, pf[0].x);  // p0 = k1, pf[0].x = length
        break;
      }
      case BendCase<THICK>::value: {  // thick sector bend: p0 = k0, pf[0] = (h, length)
        if (THICK) thick_bend<P>(q, cold, p0, pf[0].x, pf[0].y);
        break;
      }
      case RadCase<THICK>::value: {  // radiating multipole: p0 = hxl
        if (THICK) rad_multipole<P>(q, cold, slots, static_cast<int>((tag >> 8) & 0x7fu), p0, a);
        break;
      }
      case MonCase<THICK>::value: {
        if (THICK) monitor_store<P>(q, cold, p0, a.n_part);
        break;
      }
      case PolyCase<THICK>::value: {  // polygon aperture: (record bytes - header) / 16 vertices
        if (THICK) limit_polygon<P>(q, cold, slots, static_cast<int>(((tag >> 16) - sizeof(RecHdr)) / 16), elem, turns_done, a);
        break;
      }
      default:  // ... and every other combination (misaligned magnets, lone leading drifts) at run time
        if ((tag & TAG_TYPE_MASK) == TAG_MULT || (tag & TAG_TYPE_MASK) == TAG_CMULT)
          multipole_record<P, -1, -1>(q, cold, slots, pf, tag, p0);
        else if (THICK && (tag & 0xffu) == TAG_QUAD)  // instantiations whose QuadCase label is parked
          thick_quadrupole<P>(q, cold, p0, pf[0].x);
        break;
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
// (CTAs are at most 256 threads: xt_api.cu)
template <int P>
struct RegBudget {
  static constexpr int value = P == 1 ? 64 : (P == 2 ? 80 : (P == 3 ? XT_REGS3 : XT_REGS4));
};

// Shared memory: [0,16) two mbarriers; [128, 128 + 8*kPitch*blockDim) cold per-thread rows;
// then staging buffer 0 (and buffer 1 for multi-chunk lattices), 128-byte aligned, and 64
// spare bytes (the Horner loop prefetches one coefficient pair past the record it is in).
template <int P, bool THICK>
__global__ void __maxnreg__(RegBudget<P>::value) xt_track_kernel(const TrackArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  const uint32_t bar0 = smem_addr(smem);
  Cold<P> cold;
  cold.row = reinterpret_cast<double *>(smem + 128) + static_cast<uint32_t>(Cold<P>::kPitch) * threadIdx.x;
  cold.stride = static_cast<int>(blockDim.x);
  unsigned char *const buf0 =
      smem + 128 + ((static_cast<uint32_t>(8 * Cold<P>::kPitch) * blockDim.x + 127u) & ~127u);

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
      refresh_cached<P>(cold, j, opd, b, t, a.igam2);
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
  int64_t turns_done = 0;
  if (single) {
    // Whole lattice resident in buffer 0: warps run free, no CTA-level synchronisation.
    if (threadIdx.x == 0) {
      const ChunkDesc d = a.chunks[0];
      tma_load_chunk(bar0, smem_addr(buf0), a.image + d.offset, d.nbytes);
    }
    mbar_wait(bar0, 0);
    for (; turns_done < a.n_turns; ++turns_done) {
      if (!__any_sync(0xffffffffu, q.alive != 0)) break;
      track_chunk<P, THICK>(q, buf0, cold, turns_done, a);
    }
  } else {
    // A stage = stage_chunks consecutive chunks = one bulk copy into one buffer.
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
    const int64_t total = a.n_turns * n_stages;
    int64_t gidx = 0;  // global stage counter: buffer = gidx & 1, phase parity = (gidx >> 1) & 1
    int32_t c = 0;
    bool any = true;
    while (gidx < total) {
      if (threadIdx.x == 0 && gidx + 1 < total) {
        // buffer (gidx+1)&1 was released by the __syncthreads_or that ended iteration gidx-1
        load_stage((c + 1 == n_stages) ? 0 : c + 1, static_cast<uint32_t>((gidx + 1) & 1));
      }
      const uint32_t cb = static_cast<uint32_t>(gidx & 1);
      mbar_wait(bar0 + 8 * cb, static_cast<uint32_t>((gidx >> 1) & 1));
      if (__any_sync(0xffffffffu, q.alive != 0)) {
        const int32_t n_sub = (c * m + m < a.n_chunks ? m : a.n_chunks - c * m);
        const unsigned char *rp = buf0 + static_cast<size_t>(cb) * stage_bytes;
        for (int32_t k = 0; k < n_sub; ++k) rp = track_chunk<P, THICK>(q, rp, cold, turns_done, a);
      }
      ++gidx;
      if (++c == n_stages) {
        c = 0;
        ++turns_done;  // T: turn completed
      }
      any = __syncthreads_or(q.alive != 0 ? 1 : 0) != 0;
      if (!any) break;
    }
    if (!any && gidx < total) {
      // every particle of the CTA is lost: drain the copy still in flight before exiting
      mbar_wait(bar0 + 8 * static_cast<uint32_t>(gidx & 1), static_cast<uint32_t>((gidx >> 1) & 1));
    }
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

template <int P, bool THICK>
int launch_track_pt(const TrackArgs &a, const xt_lattice *lat, int block, cudaStream_t st) {
  const size_t cold_bytes = (static_cast<size_t>(8 * Cold<P>::kPitch) * block + 127) & ~static_cast<size_t>(127);
  // per device, so set on every launch (a few microseconds against launches of milliseconds to seconds)
  XT_CUDA(cudaFuncSetAttribute(xt_track_kernel<P, THICK>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  // the kernel has no use for L1 (every hot read is a shared-memory broadcast)
  XT_CUDA(cudaFuncSetAttribute(xt_track_kernel<P, THICK>, cudaFuncAttributePreferredSharedMemoryCarveout,
                               cudaSharedmemCarveoutMaxShared));
  const int64_t cap = static_cast<int64_t>(block) * P;
  const int64_t need = (a.n_part + cap - 1) / cap;
  const int64_t grid = ((need + a.grid_quantum - 1) / a.grid_quantum) * a.grid_quantum;
  if (grid > 2147483647LL) {
    set_error("xt_track: too many particles for one launch");
    return XT_ERR_INVALID_ARG;
  }
  // Staging depth: as many chunks per bulk copy (fewer CTA-wide barriers per turn) as shared memory
  // allows without taking a resident CTA away.
  cudaFuncAttributes fa;
  XT_CUDA(cudaFuncGetAttributes(&fa, xt_track_kernel<P, THICK>));
  int64_t resident = 65536 / (static_cast<int64_t>(fa.numRegs > 0 ? fa.numRegs : 128) * block);
  if (resident > grid / a.grid_quantum) resident = grid / a.grid_quantum;
  if (resident < 1) resident = 1;
  TrackArgs b = a;
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
  xt_track_kernel<P, THICK><<<static_cast<unsigned>(grid), block, smem, st>>>(b);
  count_launch();
  XT_CUDA(cudaGetLastError());
  return XT_OK;
}

// Lattices with thick elements take the instantiation that has their maps compiled in.
template <int P>
int launch_track_p(const TrackArgs &a, const xt_lattice *lat, int block, cudaStream_t st) {
  return lat->extended ? launch_track_pt<P, true>(a, lat, block, st) : launch_track_pt<P, false>(a, lat, block, st);
}

}  // namespace

int set_monitor_base(double *d_rows, cudaStream_t st) {
  XT_CUDA(cudaMemcpyToSymbolAsync(g_monitor_rows, &d_rows, sizeof(double *), 0, cudaMemcpyHostToDevice, st));
  return XT_OK;
}

int launch_track(const xt_lattice *lat, const xt_particles &p, int64_t n_part, const int64_t *d_n_active,
                 int64_t n_turns, int block, int ppt, cudaStream_t st) {
  if (n_part <= 0 || n_turns <= 0) return XT_OK;
  TrackArgs a;
  a.image = lat->d_image;
  a.chunks = lat->d_chunks;
  a.s_table = lat->d_s_table;
  a.n_active = d_n_active;
  a.p = p;
  a.n_part = n_part;
  a.n_turns = n_turns;
  a.n_chunks = static_cast<int32_t>(lat->info.n_chunks);
  a.chunk_bytes = static_cast<uint32_t>(lat->info.chunk_bytes);
  a.grid_quantum = lat->n_sm > 0 ? lat->n_sm : 1;
  a.beta0 = lat->k.beta0;
  a.tib = lat->k.tib;
  a.igam2 = lat->k.igam2;
  switch (ppt) {
    case 1:
      return launch_track_p<1>(a, lat, block, st);
    case 2:
      return launch_track_p<2>(a, lat, block, st);
    case 3:
      return launch_track_p<3>(a, lat, block, st);
    case 4:
      return launch_track_p<4>(a, lat, block, st);
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
