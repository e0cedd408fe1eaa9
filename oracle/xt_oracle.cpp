// =====================================================================================
// xt_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-threaded FP64 CPU tracker that DEFINES what the CUDA path must
// compute.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load this library.  It shares no code, header, table or
// constant generator with paper_2310_00317_b200/ (it has its own parser of the packed
// lattice buffer and its own particle struct) and must be compiled with
//     g++ -O2 -ffp-contract=off      (no FMA contraction, no fast-math)
// so that every expression below is evaluated exactly in the order written.
//
// What it follows.  The paper (PAPER.md = /root/reference/PAPER.md at survey time)
// prints no equations.  It states the structure:
//   * PAPER.md:70  "The beam line is represented as a sequence of ... objects ... each
//                   corresponding to an accelerator element ... (e.g. magnets, cavities,
//                   aperture restrictions ...)"; tilts and misalignments "are handled as
//                   changes of the reference system"; "multipolar errors".
//   * PAPER.md:72  "a 'thin' lattice integration method is adopted" (Sixtrack lineage;
//                   thin-lens formalism, ref [13] PAPER.md:255).
//   * PAPER.md:74  one kernel tracks "the entire beamline"  -> per particle: turns x elements.
//   * PAPER.md:178 aperture elements "check the particle positions with respect to the
//                   defined aperture and stop the tracking for the particles found to be outside".
//   * PAPER.md:184 non-collective tracking of different particles is independent.
// The maps themselves are the standard thin-lens symplectic maps of that formalism, in the
// reading fixed by SURVEY.md §8(c) / DESIGN.md §5 (every "paper is silent" point is listed
// there).  Since the map sequence IS the definition, this file is the algorithm written
// out element by element, turn by turn; no blocking, fusion or reordering.
//
// Pins (tests/test_oracle_pins.py, all -m "not gpu"): P1 exact-drift closed form in
// 60-digit arithmetic; P2 thin-FODO one-cell matrix / tune (closed form); P3 symplecticity
// of the one-turn Jacobian; P4 reversibility; P5 worked examples W1/W2 (60-digit textbook
// evaluation, tests/golden/); P6 Horner vs direct complex power sum; P7 Courant-Snyder
// invariant; P8 aperture edges; P9 structural invariants; P10 energy identities;
// small-amplitude synchrotron tune for the cavity; P13 thick quadrupole: second-order limit of
// thin slices (+ cubic paraxial residual), closed-form matrix, symplecticity, reversibility.
// P14 thick sector bend ('expanded'): second-order limit of thin curved-dipole slices, textbook
// matrix and dispersion, symplecticity, reversibility; P15 LimitPolygon (even-odd rule): half-plane
// test on convex polygons, union of rectangles, LimitRect on four corners
// (tests/test_oracle_refine_pins.py; P16 there pins oracle/refine.py, which tracks with this file);
// P21 mean synchrotron radiation in a thin multipole: U0 of an isomagnetic ring, scaling laws, vertical
// damping rate U0/2E, proton limit (tests/test_oracle_radiation_pins.py).
// =====================================================================================
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

constexpr double C_LIGHT = 299792458.0;       // m/s (exact, SI)
constexpr double PI = 3.14159265358979323846264338327950288;
constexpr int MAX_ORDER = 20;

enum ElemType : uint32_t {
  MARKER = 0, DRIFT = 1, MULTIPOLE = 2, CAVITY = 3,
  SROTATION = 4, XYSHIFT = 5, LIMITRECT = 6, LIMITELLIPSE = 7, QUADRUPOLE = 8, BEND = 9,
  LIMITPOLYGON = 10, RADMULTIPOLE = 12   // 11 is internal to the CUDA library
};

struct Element {
  uint32_t type = 0;
  int order = 0;
  double s_pos = 0.0;           // s at the element entrance (sum of preceding drift lengths)
  // DRIFT
  double length = 0.0;
  // MULTIPOLE: c[n] = knl[n]/n!, sn[n] = ksl[n]/n!;  with curvature c[0] = knl[0] - hxl
  std::vector<double> c, sn;
  double hxl = 0.0, wf = 0.0;
  // CAVITY
  double lag_rad = 0.0, kz = 0.0, vn = 0.0;
  // SROTATION
  double cz = 1.0, sz = 0.0;
  // XYSHIFT
  double dx = 0.0, dy = 0.0;
  // LIMITRECT
  double min_x = 0.0, max_x = 0.0, min_y = 0.0, max_y = 0.0;
  // LIMITELLIPSE
  double a = 0.0, b = 0.0, a2 = 0.0, b2 = 0.0, a2b2 = 0.0;
  // QUADRUPOLE (thick): k1, length
  double k1 = 0.0;
  // BEND (thick sector bend): k0, h, length; model 0 = 'expanded', 1 = 'full'
  double k0 = 0.0, h = 0.0;
  int model = 0;
  // LIMITPOLYGON: vertices (vx[i], vy[i]), closed
  std::vector<double> vx, vy;
  // RADMULTIPOLE: as MULTIPOLE (c[0] folded, wf from the raw knl[0]), plus krad = (2/3) r0 (beta0 gamma0)^3
  double krad = 0.0;
};

struct Lattice {
  double p0c = 0, mass0 = 0, q0 = 0;
  double beta0 = 0, gamma0 = 0;
  double tib = 0;      // 2/beta0
  double igam2 = 0;    // 1/gamma0^2
  std::vector<Element> el;
};

double factorial(int n) {               // exact in FP64 for n <= 22
  double f = 1.0;
  for (int i = 2; i <= n; ++i) f = f * static_cast<double>(i);
  return f;
}

// Parse the packed lattice buffer (layout: xt_inputs/packed.py docstring).  Own parser;
// the CUDA library has a different one.  Returns 0 or a negative error code.
int parse(const void* packed, size_t nbytes, Lattice& L) {
  const unsigned char* p = static_cast<const unsigned char*>(packed);
  if (!p || nbytes < 48) return -2;
  if (std::memcmp(p, "XTLAT001", 8) != 0) return -2;
  uint32_t version, n_el;
  uint64_t total;
  std::memcpy(&version, p + 8, 4);
  std::memcpy(&n_el, p + 12, 4);
  std::memcpy(&L.p0c, p + 16, 8);
  std::memcpy(&L.mass0, p + 24, 8);
  std::memcpy(&L.q0, p + 32, 8);
  std::memcpy(&total, p + 40, 8);
  if (version != 1 || total != nbytes) return -2;
  if (!(L.p0c > 0.0) || !(L.mass0 > 0.0) || !std::isfinite(L.p0c) || !std::isfinite(L.mass0) ||
      !std::isfinite(L.q0))
    return -2;
  // Reference particle: E0 = sqrt(p0c^2 + mass0^2), beta0 = p0c/E0, gamma0 = E0/mass0.
  const double e0 = std::sqrt(L.p0c * L.p0c + L.mass0 * L.mass0);
  L.beta0 = L.p0c / e0;
  L.gamma0 = e0 / L.mass0;
  L.tib = 2.0 / L.beta0;
  L.igam2 = 1.0 / (L.gamma0 * L.gamma0);

  size_t off = 48;
  double s = 0.0;
  auto rd = [&](double& v) -> bool {
    if (off + 8 > nbytes) return false;
    std::memcpy(&v, p + off, 8);
    off += 8;
    return std::isfinite(v);
  };
  L.el.clear();
  // every record is at least 8 bytes: a count the buffer cannot hold is a truncated buffer (found by the
  // ASan run of tests/test_sanitizers.py: a 48-byte buffer announcing 2^32 - 1 elements reserved 1.2 TB)
  if (n_el > (nbytes - 48) / 8) return -2;
  L.el.reserve(n_el);
  for (uint32_t i = 0; i < n_el; ++i) {
    if (off + 8 > nbytes) return -2;
    Element e;
    uint32_t aux;
    std::memcpy(&e.type, p + off, 4);
    std::memcpy(&aux, p + off + 4, 4);
    off += 8;
    e.s_pos = s;
    switch (e.type) {
      case MARKER: break;
      case DRIFT:
        if (!rd(e.length)) return -2;
        s = s + e.length;
        break;
      case MULTIPOLE: {
        if (aux > static_cast<uint32_t>(MAX_ORDER)) return -2;
        e.order = static_cast<int>(aux);
        double length;
        if (!rd(e.hxl) || !rd(length)) return -2;
        std::vector<double> knl(e.order + 1), ksl(e.order + 1);
        for (int n = 0; n <= e.order; ++n) if (!rd(knl[n])) return -2;
        for (int n = 0; n <= e.order; ++n) if (!rd(ksl[n])) return -2;
        e.c.resize(e.order + 1);
        e.sn.resize(e.order + 1);
        for (int n = 0; n <= e.order; ++n) {
          e.c[n] = knl[n] / factorial(n);
          e.sn[n] = ksl[n] / factorial(n);
        }
        e.wf = 0.0;
        if (e.hxl != 0.0) {
          // Curvature folded into the dipole coefficient (cancellation-free form,
          // DESIGN.md §5 "Multipole"): -k0l + hxl(1+delta) = -(k0l - hxl) + hxl*delta.
          e.c[0] = knl[0] - e.hxl;
          if (length != 0.0) e.wf = (knl[0] * e.hxl) / length;   // weak focusing k0*h*L
        }
        break;
      }
      case CAVITY: {
        double volt, freq, lag_deg;
        if (!rd(volt) || !rd(freq) || !rd(lag_deg)) return -2;
        e.lag_rad = lag_deg * (PI / 180.0);
        e.kz = (2.0 * PI * freq) / (L.beta0 * C_LIGHT);
        e.vn = (L.q0 * volt) / L.p0c;
        break;
      }
      case SROTATION:
        if (!rd(e.cz) || !rd(e.sz)) return -2;
        break;
      case XYSHIFT:
        if (!rd(e.dx) || !rd(e.dy)) return -2;
        break;
      case LIMITRECT:
        if (!rd(e.min_x) || !rd(e.max_x) || !rd(e.min_y) || !rd(e.max_y)) return -2;
        break;
      case LIMITELLIPSE:
        if (!rd(e.a) || !rd(e.b)) return -2;
        e.a2 = e.a * e.a;
        e.b2 = e.b * e.b;
        e.a2b2 = e.a2 * e.b2;
        break;
      case QUADRUPOLE:
        if (!rd(e.k1) || !rd(e.length)) return -2;
        if (e.k1 == 0.0 || !(e.length > 0.0)) return -2;   // a zero-strength thick quadrupole is a Drift
        s = s + e.length;
        break;
      case BEND:
        if (!rd(e.k0) || !rd(e.h) || !rd(e.length)) return -2;
        if (!(e.k0 * e.h > 0.0) || !(e.length > 0.0)) return -2;   // focusing strength k0 h must be > 0
        if (aux > 1u) return -2;                                     // 0: 'expanded', 1: 'full'
        e.model = static_cast<int>(aux);
        s = s + e.length;
        break;
      case RADMULTIPOLE: {
        // Thin multipole that radiates ("mean" model; reading A22): parameters as MULTIPOLE,
        // length > 0 (the curvature of the trajectory is kick / length).
        if (aux > static_cast<uint32_t>(MAX_ORDER)) return -2;
        e.order = static_cast<int>(aux);
        if (!rd(e.hxl) || !rd(e.length)) return -2;
        if (!(e.length > 0.0)) return -2;
        e.c.resize(e.order + 1);
        e.sn.resize(e.order + 1);
        for (int n = 0; n <= e.order; ++n) { double v; if (!rd(v)) return -2; e.c[n] = v / factorial(n); }
        for (int n = 0; n <= e.order; ++n) { double v; if (!rd(v)) return -2; e.sn[n] = v / factorial(n); }
        e.wf = (e.c[0] * e.hxl) / e.length;
        e.c[0] = e.c[0] - e.hxl;      // curvature folded into the dipole coefficient, as in MULTIPOLE (cancellation-free)
        // classical radius r0 = q0^2 e^2/(4 pi eps0 m c^2), e^2/(4 pi eps0) = 1.4399645478e-9 eV m (CODATA 2018)
        const double r0 = ((L.q0 * L.q0) * 1.4399645478e-9) / L.mass0;
        const double bg0 = L.p0c / L.mass0;
        e.krad = ((2.0 / 3.0) * r0) * ((bg0 * bg0) * bg0);
        break;
      }
      case LIMITPOLYGON:
        if (aux < 3 || aux > 256) return -2;
        e.vx.resize(aux);
        e.vy.resize(aux);
        for (uint32_t n = 0; n < aux; ++n) if (!rd(e.vx[n])) return -2;
        for (uint32_t n = 0; n < aux; ++n) if (!rd(e.vy[n])) return -2;
        break;
      default: return -2;
    }
    L.el.push_back(std::move(e));
  }
  if (off != nbytes) return -2;
  return 0;
}

// Per-particle cached constants: pure functions of the stored delta, ptau; recomputed
// only after a cavity (DESIGN.md §5 "Per-particle cached constants").
struct Cached {
  double opd2, b, g, rv0v;
};

inline Cached derive_cached(const Lattice& L, double delta, double ptau) {
  Cached k;
  const double opd = 1.0 + delta;
  k.opd2 = opd * opd;
  k.b = 1.0 + L.beta0 * ptau;
  const double t = ptau * (ptau + L.tib);
  k.g = t * L.igam2;
  k.rv0v = k.b / opd;
  return k;
}

}  // namespace

extern "C" {

// Host pointers, all of length n_part.  at_element and min_margin may be NULL.
struct xo_particles {
  double *x, *px, *y, *py, *zeta, *delta, *ptau, *rpp, *rvv, *s;
  int64_t *at_turn, *state, *at_element;
  double* min_margin;   // out (if non-NULL): min over all aperture checks passed through of
                        // the distance [m] to the aperture edge (reading A3); +inf if none
};

// delta -> ptau, rpp, rvv (DESIGN.md §5 "Init helper"):
//   t = delta*(delta+2); ptau = t/(sqrt(t + 1/beta0^2) + 1/beta0)   [= sqrt((1+delta)^2 + 1/(b0 g0)^2)... energy identity]
int xo_init_derived(const void* packed, size_t nbytes, const double* delta, double* ptau,
                    double* rpp, double* rvv, int64_t n) {
  Lattice L;
  int rc = parse(packed, nbytes, L);
  if (rc) return rc;
  const double ib = 1.0 / L.beta0;
  const double ib2 = ib * ib;
  for (int64_t i = 0; i < n; ++i) {
    const double d = delta[i];
    const double t = d * (d + 2.0);
    const double pt = t / (std::sqrt(t + ib2) + ib);
    const double opd = 1.0 + d;
    const double b = 1.0 + L.beta0 * pt;
    ptau[i] = pt;
    rpp[i] = 1.0 / opd;
    rvv[i] = opd / b;
  }
  return 0;
}

// Reference-particle quantities as the oracle derives them (for tests / input scaling).
int xo_reference(const void* packed, size_t nbytes, double* beta0, double* gamma0) {
  Lattice L;
  int rc = parse(packed, nbytes, L);
  if (rc) return rc;
  *beta0 = L.beta0;
  *gamma0 = L.gamma0;
  return 0;
}

// s position (entrance) of every element; out has n_elements entries.  Returns n_elements.
int64_t xo_s_table(const void* packed, size_t nbytes, double* out, int64_t cap) {
  Lattice L;
  int rc = parse(packed, nbytes, L);
  if (rc) return rc;
  const int64_t n = static_cast<int64_t>(L.el.size());
  for (int64_t i = 0; i < n && i < cap; ++i) out[i] = L.el[i].s_pos;
  return n;
}

// Track n_part particles for n_turns turns through the whole line.
// In/out arrays as in xo_particles.  Lost particles (state == 0) are skipped entirely.
int xo_track(const void* packed, size_t nbytes, const xo_particles* P, int64_t n_part,
             int64_t n_turns) {
  if (!P || n_part < 0 || n_turns < 0) return -1;
  Lattice L;
  int rc = parse(packed, nbytes, L);
  if (rc) return rc;
  const int64_t n_el = static_cast<int64_t>(L.el.size());

  for (int64_t ip = 0; ip < n_part; ++ip) {
    double x = P->x[ip], px = P->px[ip], y = P->y[ip], py = P->py[ip];
    double zeta = P->zeta[ip], delta = P->delta[ip], ptau = P->ptau[ip];
    double rpp = P->rpp[ip], rvv = P->rvv[ip], s = P->s[ip];
    int64_t at_turn = P->at_turn[ip], state = P->state[ip];
    int64_t at_element = P->at_element ? P->at_element[ip] : 0;
    double margin = std::numeric_limits<double>::infinity();
    Cached k = derive_cached(L, delta, ptau);

    for (int64_t turn = 0; turn < n_turns && state == 1; ++turn) {
      for (int64_t ie = 0; ie < n_el && state == 1; ++ie) {
        const Element& e = L.el[ie];
        switch (e.type) {
          case MARKER: break;

          case DRIFT: {
            // Exact drift (thin-lattice integration):
            //   x += L px/pz, y += L py/pz, zeta += L (1 - (1+beta0 ptau)/pz),
            //   pz = sqrt((1+delta)^2 - px^2 - py^2),
            // with the zeta increment rewritten cancellation-free through
            //   pz^2 - b^2 = g - px^2 - py^2   (DESIGN.md §5 "Drift").
            const double t1 = px * px;
            const double pxy2 = py * py + t1;
            const double pz = std::sqrt(k.opd2 - pxy2);
            const double s1 = pz + k.b;
            const double den = pz * s1;
            const double rr = 1.0 / den;
            const double lr = e.length * rr;
            const double lpz = lr * s1;
            x = px * lpz + x;
            y = py * lpz + y;
            zeta = (k.g - pxy2) * lr + zeta;
            break;
          }

          case MULTIPOLE: {
            // Thin multipole kick ("multipolar errors", PAPER.md:72 thin maps):
            //   dpx - i dpy = -sum_n (knl[n] + i ksl[n]) (x + i y)^n / n!   by complex Horner,
            // highest order first.
            const int N = e.order;
            double re = e.c[N];
            double im = e.sn[N];
            for (int n = N - 1; n >= 0; --n) {
              const double nre = re * x + (e.c[n] - im * y);
              const double nim = re * y + (e.sn[n] + im * x);
              re = nre;
              im = nim;
            }
            px = px - re;
            py = py + im;
            if (e.hxl != 0.0) {
              // Horizontal curvature: dpx = hxl (1+delta) [the hxl*1 part is folded into c[0]],
              // weak focusing -k0 h L x, path length dzeta = -hxl x beta0/beta.
              px = e.hxl * delta + px;
              px = px - e.wf * x;
              zeta = zeta - (e.hxl * x) * k.rv0v;
            }
            break;
          }

          case RADMULTIPOLE: {
            // "Mean" synchrotron radiation ("the energy loss from the radiation is applied
            // particle by particle without accounting for quantum fluctuations"; "only for the thin lattice
            // modelling").  Reading A22.  The field of the slice bends the trajectory with
            // curvature kappa = |kick| P0/(P lpath), lpath = length (1 + h x); the classical power
            // (2/3) r0 m c^3 beta^4 gamma^4 kappa^2 over the time lpath/(beta c) takes the fraction
            //   r = (2/3) r0 (beta gamma)^3 kappa^2 lpath = krad (1+delta) kick^2 / lpath
            // of the particle's energy (beta gamma = beta0 gamma0 (1+delta)).  Half of it is taken before the
            // kick and half after; each time the energy drops, E' = E (1 - r/2), the momentum follows from
            // the energy (as behind a cavity) and px, py shrink with it: the photon leaves along the motion.
            const int N = e.order;
            double re = e.c[N];
            double im = e.sn[N];
            for (int n = N - 1; n >= 0; --n) {
              const double nre = re * x + (e.c[n] - im * y);
              const double nim = re * y + (e.sn[n] + im * x);
              re = nre;
              im = nim;
            }
            const double dpxf = (-re - e.hxl) - e.wf * x;  // the field's kick (re has the curvature folded in; weak focusing included)
            const double dpyf = im;
            const double kick2 = dpxf * dpxf + dpyf * dpyf;
            const double lpath = e.length + e.hxl * x;
            for (int half = 0; half < 2; ++half) {
              const double opd = 1.0 + delta;
              const double rh = ((0.5 * e.krad) * (opd * kick2)) / lpath;
              ptau = ptau - rh * (ptau + 1.0 / L.beta0);
              const double t = ptau * (ptau + L.tib);
              delta = t / (std::sqrt(t + 1.0) + 1.0);
              const double opd1 = 1.0 + delta;
              const double f = opd1 / opd;
              px = px * f;
              py = py * f;
              rpp = 1.0 / opd1;
              const double b = 1.0 + L.beta0 * ptau;
              rvv = opd1 / b;
              k.opd2 = opd1 * opd1;
              k.b = b;
              k.g = t * L.igam2;
              k.rv0v = b / opd1;
              if (half == 0) {                             // the thin kick itself, in the arithmetic of MULTIPOLE
                px = px - re;
                py = py + im;
                px = e.hxl * delta + px;
                px = px - e.wf * x;
                zeta = zeta - (e.hxl * x) * k.rv0v;
              }
            }
            break;
          }

          case QUADRUPOLE: {
            // Thick quadrupole ("'Thick' maps for ... quadrupole magnets"; reading A18):
            // exact flow of H = (px^2 + py^2)/(2(1+delta)) + (k1/2)(x^2 - y^2) over the length L.
            // With w = sqrt(|k1|/(1+delta)) the focusing plane (u, pu) turns by the angle w L,
            //   u' = u cos + pu sin/((1+delta) w),   pu' = pu cos - (1+delta) w u sin,
            // the other one (v, pv) follows cosh / sinh, and the path length is
            //   zeta' = zeta + L (1 - beta0/beta) - (beta0/beta)/(2 (1+delta)^2) int_0^L (px^2 + py^2) ds,
            // the first term written cancellation-free as L g/((1+delta)((1+delta) + b)).
            const double opd = 1.0 + delta;
            const double rk = e.k1 / opd;
            const double w = std::sqrt(std::fabs(rk));
            const double wl = w * e.length;
            const double cs = std::cos(wl), sn = std::sin(wl);
            const double ch = std::cosh(wl), sh = std::sinh(wl);
            const double ow = opd * w;
            const double iw = 1.0 / ow;
            const bool focus_x = rk > 0.0;
            const double u = focus_x ? x : y, pu = focus_x ? px : py;
            const double v = focus_x ? y : x, pv = focus_x ? py : px;
            const double au = ow * u;
            const double av = ow * v;
            const double u1 = u * cs + (pu * iw) * sn;
            const double pu1 = pu * cs - au * sn;
            const double v1 = v * ch + (pv * iw) * sh;
            const double pv1 = pv * ch + av * sh;
            const double hl = 0.5 * e.length;
            const double h2w = 0.5 / w;
            const double pu2 = pu * pu, au2 = au * au, pv2 = pv * pv, av2 = av * av;
            const double i_f = ((pu2 + au2) * hl + ((pu2 - au2) * (sn * cs)) * h2w) - ((au * pu) * (sn * sn)) / w;
            const double i_d = ((pv2 - av2) * hl + ((pv2 + av2) * (sh * ch)) * h2w) + ((av * pv) * (sh * sh)) / w;
            zeta = (zeta + e.length * (k.g / (opd * (opd + k.b)))) - (k.rv0v / (2.0 * k.opd2)) * (i_f + i_d);
            if (focus_x) { x = u1; px = pu1; y = v1; py = pv1; }
            else         { y = u1; py = pu1; x = v1; px = pv1; }
            break;
          }

          case BEND: {
            if (e.model == 1) {
              // Thick sector bend, 'full' model ("a 'full' map, which is appropriate for small
              // accelerators [12]"; reading A23): the exact map of a charge in the uniform field k0 seen from
              // the frame that follows the arc of curvature h -- the helix, cut by the exit plane.  With
              // pz = sqrt((1+delta)^2 - px^2 - py^2), theta = h L and C = pz - k0 (1/h + x):
              //   px' = px cos(theta) + C sin(theta)
              //   x'  = (h pz' - dpx'/ds - k0)/(h k0),  dpx'/ds = h (C cos(theta) - px sin(theta))
              //   y'  = y + py (theta + D)/k0,  D = asin(px/ph) - asin(px'/ph),  ph^2 = (1+delta)^2 - py^2
              //   zeta' = zeta + L - (1 + beta0 ptau)(theta + D)/k0          (path length (1+delta)(theta + D)/k0)
              // evaluated in a form without cancellation (the reference particle of a matched bend has every
              // term below exactly zero): pz - 1 = (delta(delta+2) - px^2 - py^2)/(pz + 1),
              // C = (pz - 1) - (k0 - h)/h - k0 x,  1 - cos(theta) = 2 sin^2(theta/2),
              // pz' - pz = -(px' - px)(px' + px)/(pz' + pz), which turn x' into
              //   x' = x + [px sin + (1 - cos) C - (px' - px)(px + px')/(pz' + pz)]/k0
              // and L - (1 + beta0 ptau) theta/k0 into ((k0 - h) - h beta0 ptau) L/k0.
              const double t1 = px * px;
              const double pxy2 = py * py + t1;
              const double pz = std::sqrt(k.opd2 - pxy2);
              const double dpz = (delta * (delta + 2.0) - pxy2) / (pz + 1.0);
              const double eps = (e.k0 - e.h) / e.h;
              const double cc = (dpz - eps) - e.k0 * x;
              const double th = e.h * e.length;
              const double sn = std::sin(th);
              const double sh = std::sin(0.5 * th);
              const double c1 = 2.0 * (sh * sh);
              const double dpx = cc * sn - px * c1;
              const double px1 = px + dpx;
              const double ph2 = k.opd2 - py * py;
              const double pz1 = std::sqrt(ph2 - px1 * px1);
              const double num = (px * sn + c1 * cc) - (dpx * (px + px1)) / (pz1 + pz);
              const double iph = 1.0 / std::sqrt(ph2);
              const double dd = std::asin(px * iph) - std::asin(px1 * iph);
              x = num / e.k0 + x;
              y = (py * (th + dd)) / e.k0 + y;
              zeta = (zeta + (((e.k0 - e.h) - e.h * (L.beta0 * ptau)) * e.length) / e.k0) - (k.b * dd) / e.k0;
              px = px1;
              break;
            }
            // Thick sector bend, 'expanded' model ("the bend can be 'full' or 'expanded'";
            // reading A19): exact flow of
            //   H = (px^2 + py^2)/(2(1+delta)) - h x (1+delta) + k0 x + (k0 h/2) x^2
            // (the thin curved multipole of this file, smeared over the arc length L).  With
            // K = k0 h, w = sqrt(K/(1+delta)) and the equilibrium offset xe = (h (1+delta) - k0)/K:
            //   x' - xe = (x - xe) cos + px sin/((1+delta) w),  px' = px cos - (1+delta) w (x - xe) sin,
            //   y' = y + L py/(1+delta),
            //   zeta' = zeta + L (1 - beta0/beta) - (beta0/beta) h int x ds
            //           - (beta0/beta)/(2 (1+delta)^2) (int px^2 ds + L py^2).
            const double opd = 1.0 + delta;
            const double kk = e.k0 * e.h;
            const double w = std::sqrt(kk / opd);
            const double wl = w * e.length;
            const double cs = std::cos(wl), sn = std::sin(wl);
            const double c1 = 1.0 - cs;
            const double ow = opd * w;
            const double fw = (e.h * opd - e.k0) / w;            // (1+delta) w xe: the offset enters only through it
            const double a = ow * x - fw;                         // (1+delta) w (x - xe)
            const double pw = px / ow;
            const double x1 = (x * cs + pw * sn) + (fw * c1) / ow;
            const double px1 = px * cs - a * sn;
            const double y1 = (e.length * py) / opd + y;
            const double ix = ((x * sn) / w + (pw * c1) / w) + (fw / ow) * (e.length - sn / w);   // int x ds
            const double px2 = px * px, a2 = a * a;
            const double ip = ((px2 + a2) * (0.5 * e.length) + ((px2 - a2) * (sn * cs)) * (0.5 / w)) -
                              ((a * px) * (sn * sn)) / w;                                     // int px^2 ds
            zeta = ((zeta + e.length * (k.g / (opd * (opd + k.b)))) - (k.rv0v * e.h) * ix) -
                   (k.rv0v / (2.0 * k.opd2)) * (ip + e.length * (py * py));
            x = x1; px = px1; y = y1;
            break;
          }

          case CAVITY: {
            // Thin RF cavity: energy kick, transverse normalised momenta unchanged.
            const double phase = e.lag_rad - e.kz * zeta;
            ptau = e.vn * std::sin(phase) + ptau;
            const double t = ptau * (ptau + L.tib);
            delta = t / (std::sqrt(t + 1.0) + 1.0);     // = sqrt(1+t) - 1 without cancellation
            const double opd = 1.0 + delta;
            rpp = 1.0 / opd;
            const double b = 1.0 + L.beta0 * ptau;
            rvv = opd / b;
            k.opd2 = opd * opd;
            k.b = b;
            k.g = t * L.igam2;
            k.rv0v = b / opd;
            break;
          }

          case SROTATION: {
            // Rotation of the reference system about s ("tilts").
            const double nx = e.cz * x + e.sz * y;
            const double ny = e.cz * y - e.sz * x;
            const double npx = e.cz * px + e.sz * py;
            const double npy = e.cz * py - e.sz * px;
            x = nx; y = ny; px = npx; py = npy;
            break;
          }

          case XYSHIFT:
            // Transverse shift of the reference system ("misalignments").
            x = x - e.dx;
            y = y - e.dy;
            break;

          case LIMITRECT: {
            // PAPER.md:178; edges inclusive, NaN -> lost (reading A3, A4).
            const bool inside = (x >= e.min_x) && (x <= e.max_x) && (y >= e.min_y) && (y <= e.max_y);
            double m = std::fmin(std::fmin(x - e.min_x, e.max_x - x), std::fmin(y - e.min_y, e.max_y - y));
            m = std::fabs(m);
            if (m < margin) margin = m;
            if (!inside) { state = 0; at_element = ie; s = e.s_pos; }
            break;
          }

          case LIMITELLIPSE: {
            const double tt = (x * x) * e.b2 + (y * y) * e.a2;
            const bool inside = (tt <= e.a2b2);
            double m = std::fabs(std::sqrt((x * x) / e.a2 + (y * y) / e.b2) - 1.0) * std::fmin(e.a, e.b);
            if (m < margin) margin = m;
            if (!inside) { state = 0; at_element = ie; s = e.s_pos; }
            break;
          }

          case LIMITPOLYGON: {
            // PAPER.md:178 "polygonal" aperture (reading A20): even-odd rule.  The half line from the
            // particle towards +x crosses edge (j -> i) iff the edge's ends lie on different sides of the
            // horizontal through the particle and the crossing point is to the right of it; an odd
            // number of crossings means inside.  NaN coordinates cross nothing: lost (reading A4).
            const size_t nv = e.vx.size();
            bool inside = false;
            double m = INFINITY;
            for (size_t i = 0, j = nv - 1; i < nv; j = i, ++i) {
              const double xi = e.vx[i], yi = e.vy[i], xj = e.vx[j], yj = e.vy[j];
              if ((yi > y) != (yj > y)) {
                const double xc = ((xj - xi) * (y - yi)) / (yj - yi) + xi;
                if (x < xc) inside = !inside;
              }
              // distance to the edge (margin bookkeeping only)
              const double ex = xj - xi, ey = yj - yi;
              const double l2 = ex * ex + ey * ey;
              double t = l2 > 0.0 ? ((x - xi) * ex + (y - yi) * ey) / l2 : 0.0;
              t = std::fmin(1.0, std::fmax(0.0, t));
              const double qx = x - (xi + t * ex), qy = y - (yi + t * ey);
              const double d = std::sqrt(qx * qx + qy * qy);
              if (d < m) m = d;
            }
            if (m < margin) margin = m;
            if (!inside) { state = 0; at_element = ie; s = e.s_pos; }
            break;
          }
        }
      }
      if (state == 1) {      // turn completed
        at_turn = at_turn + 1;
        s = 0.0;
      }
    }

    P->x[ip] = x; P->px[ip] = px; P->y[ip] = y; P->py[ip] = py;
    P->zeta[ip] = zeta; P->delta[ip] = delta; P->ptau[ip] = ptau;
    P->rpp[ip] = rpp; P->rvv[ip] = rvv; P->s[ip] = s;
    P->at_turn[ip] = at_turn; P->state[ip] = state;
    if (P->at_element) P->at_element[ip] = at_element;
    if (P->min_margin) P->min_margin[ip] = margin;
  }
  return 0;
}

}  // extern "C"
