// Twiss from tracking, 4-D ("Twiss module"):
//   1. "the closed orbit is found by a root finder" applied to the one-turn map,
//   2. "the Jacobian matrix of the one-turn map is computed by central differences" of
//      tracked particles,
//   3. the linear optics follows from that matrix (here: the uncoupled reading per plane,
//      cos mu = (M11 + M22)/2, beta = M12/sin mu, alpha = (M11 - M22)/(2 sin mu)).
// The tracker is the inner loop of everything: each Newton step is ONE xt_track launch of
// nine particles (the orbit and +-h along x, px, y, py) through the whole line; only the
// 4 x 4 linear algebra runs on the host.
#include <cmath>

#include <algorithm>
#include <complex>
#include <vector>

#include "xt_internal.h"
#include "xt_line.h"

namespace xt {
namespace {

constexpr int kProbe = 9;      // orbit + 2 x 4 displaced particles
constexpr int kArr = 14;       // device arrays of the probe ensemble
constexpr double kStep[4] = {1e-6, 1e-8, 1e-6, 1e-8};  // central-difference steps: x, px, y, py

struct Probe {
  double *d[10] = {};    // x px y py zeta delta ptau rpp rvv s
  int64_t *i[4] = {};    // at_turn state particle_id at_element
  void *block = nullptr;
};

int solve4(double a[4][5]) {  // Gaussian elimination with partial pivoting on [A | b]
  for (int c = 0; c < 4; ++c) {
    int piv = c;
    for (int r = c + 1; r < 4; ++r)
      if (std::fabs(a[r][c]) > std::fabs(a[piv][c])) piv = r;
    if (a[piv][c] == 0.0) return -1;
    if (piv != c)
      for (int k = 0; k < 5; ++k) std::swap(a[piv][k], a[c][k]);
    for (int r = c + 1; r < 4; ++r) {
      const double f = a[r][c] / a[c][c];
      for (int k = c; k < 5; ++k) a[r][k] -= f * a[c][k];
    }
  }
  for (int r = 3; r >= 0; --r) {
    double s = a[r][4];
    for (int k = r + 1; k < 4; ++k) s -= a[r][k] * a[k][4];
    a[r][4] = s / a[r][r];
  }
  return 0;
}

// One launch: track the orbit z and its eight neighbours for one turn.
// out[0] = image of z, jac = central-difference Jacobian (row-major).  Returns XT_ERR_UNSTABLE
// if any of the nine particles is lost or non-finite.
int one_turn_and_jacobian(const xt_lattice *lat, const Probe &pr, const double z[4], double delta0, double out[4],
                          double jac[16], cudaStream_t st) {
  double h_x[4][kProbe];
  for (int c = 0; c < 4; ++c)
    for (int k = 0; k < kProbe; ++k) h_x[c][k] = z[c];
  for (int c = 0; c < 4; ++c) {
    h_x[c][1 + 2 * c] += kStep[c];
    h_x[c][2 + 2 * c] -= kStep[c];
  }
  double zeros[kProbe] = {}, deltas[kProbe];
  int64_t ones[kProbe], izeros[kProbe] = {};
  for (int k = 0; k < kProbe; ++k) {
    deltas[k] = delta0;
    ones[k] = 1;
  }
  const size_t nb = kProbe * 8;
  for (int c = 0; c < 4; ++c) XT_CUDA(cudaMemcpyAsync(pr.d[c], h_x[c], nb, cudaMemcpyHostToDevice, st));
  XT_CUDA(cudaMemcpyAsync(pr.d[4], zeros, nb, cudaMemcpyHostToDevice, st));   // zeta
  XT_CUDA(cudaMemcpyAsync(pr.d[5], deltas, nb, cudaMemcpyHostToDevice, st));  // delta
  XT_CUDA(cudaMemcpyAsync(pr.d[9], zeros, nb, cudaMemcpyHostToDevice, st));   // s
  XT_CUDA(cudaMemcpyAsync(pr.i[0], izeros, nb, cudaMemcpyHostToDevice, st));  // at_turn
  XT_CUDA(cudaMemcpyAsync(pr.i[1], ones, nb, cudaMemcpyHostToDevice, st));    // state
  XT_CUDA(cudaMemcpyAsync(pr.i[3], izeros, nb, cudaMemcpyHostToDevice, st));  // at_element
  xt_particles p{};
  p.x = pr.d[0];
  p.px = pr.d[1];
  p.y = pr.d[2];
  p.py = pr.d[3];
  p.zeta = pr.d[4];
  p.delta = pr.d[5];
  p.ptau = pr.d[6];
  p.rpp = pr.d[7];
  p.rvv = pr.d[8];
  p.s = pr.d[9];
  p.at_turn = pr.i[0];
  p.state = pr.i[1];
  p.particle_id = nullptr;
  p.at_element = pr.i[3];
  int rc = launch_init_derived(lat, p, kProbe, st);
  if (rc != XT_OK) return rc;
  rc = xt_track(lat, &p, kProbe, 1, st);
  if (rc != XT_OK) return rc;
  double r[4][kProbe];
  int64_t state[kProbe];
  for (int c = 0; c < 4; ++c) XT_CUDA(cudaMemcpyAsync(r[c], pr.d[c], nb, cudaMemcpyDeviceToHost, st));
  XT_CUDA(cudaMemcpyAsync(state, pr.i[1], nb, cudaMemcpyDeviceToHost, st));
  XT_CUDA(cudaStreamSynchronize(st));
  for (int k = 0; k < kProbe; ++k) {
    bool ok = state[k] == 1;
    for (int c = 0; c < 4; ++c) ok = ok && std::isfinite(r[c][k]);
    if (!ok) {
      set_error("xt_twiss4d: a probe particle was lost or became non-finite (orbit outside the aperture?)");
      return XT_ERR_UNSTABLE;
    }
  }
  for (int row = 0; row < 4; ++row) {
    out[row] = r[row][0];
    for (int c = 0; c < 4; ++c) jac[4 * row + c] = (r[row][1 + 2 * c] - r[row][2 + 2 * c]) / (2.0 * kStep[c]);
  }
  return XT_OK;
}

}  // namespace
}  // namespace xt

static int xt_twiss4d_impl(const xt_lattice *lat, double delta0, const double *guess4, xt_twiss4d_result *out,
                          void *cuda_stream) {
  using namespace xt;
  if (!lat || !out || !std::isfinite(delta0)) {
    set_error("xt_twiss4d: NULL lattice / result or non-finite delta0");
    return XT_ERR_INVALID_ARG;
  }
  if (const int rc_dev = check_device(lat, "xt_twiss4d")) return rc_dev;  // before any allocation or launch
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  Probe pr;
  const size_t pitch = 256;  // bytes per array (9 x 8 = 72 used)
  XT_CUDA(cudaMalloc(&pr.block, pitch * kArr));
  unsigned char *base = static_cast<unsigned char *>(pr.block);
  for (int k = 0; k < 10; ++k) pr.d[k] = reinterpret_cast<double *>(base + pitch * k);
  for (int k = 0; k < 4; ++k) pr.i[k] = reinterpret_cast<int64_t *>(base + pitch * (10 + k));
  auto done = [&](int code) {
    cudaFree(pr.block);
    return code;
  };

  double z[4] = {0.0, 0.0, 0.0, 0.0};
  if (guess4)
    for (int c = 0; c < 4; ++c) z[c] = guess4[c];
  xt_twiss4d_result res{};
  double img[4], jac[16];
  int rc = XT_OK;
  bool converged = false;
  for (int it = 0; it < 25; ++it) {  // Twiss step 1: Newton on f(z) - z = 0
    if ((rc = one_turn_and_jacobian(lat, pr, z, delta0, img, jac, st)) != XT_OK) return done(rc);
    double a[4][5];
    for (int r = 0; r < 4; ++r) {
      for (int c = 0; c < 4; ++c) a[r][c] = jac[4 * r + c] - (r == c ? 1.0 : 0.0);
      a[r][4] = -(img[r] - z[r]);
    }
    if (solve4(a) != 0) {
      set_error("xt_twiss4d: one-turn matrix minus identity is singular (integer tune?)");
      return done(XT_ERR_UNSTABLE);
    }
    double step = 0.0;
    for (int c = 0; c < 4; ++c) {
      z[c] += a[c][4];
      step = std::fmax(step, std::fabs(a[c][4]));
    }
    res.iterations = it + 1;
    if (step < 1e-13) {
      converged = true;
      break;
    }
  }
  if (!converged) {
    set_error("xt_twiss4d: closed-orbit search did not converge in 25 Newton steps");
    return done(XT_ERR_UNSTABLE);
  }
  // Twiss step 2: the Jacobian at the closed orbit; step 3: uncoupled optics per plane
  if ((rc = one_turn_and_jacobian(lat, pr, z, delta0, img, jac, st)) != XT_OK) return done(rc);
  for (int c = 0; c < 4; ++c) res.co[c] = z[c];
  for (int k = 0; k < 16; ++k) res.m[k] = jac[k];
  res.stable = 1;
  double *bet[2] = {&res.betx, &res.bety}, *alf[2] = {&res.alfx, &res.alfy};
  double *mu[2] = {&res.mux, &res.muy}, *q[2] = {&res.qx_frac, &res.qy_frac};
  for (int pl = 0; pl < 2; ++pl) {
    const int i = 2 * pl;
    const double m11 = jac[4 * i + i], m12 = jac[4 * i + i + 1], m22 = jac[4 * (i + 1) + i + 1];
    const double cosmu = 0.5 * (m11 + m22);
    if (!(std::fabs(cosmu) < 1.0)) {
      res.stable = 0;
      *bet[pl] = *alf[pl] = *mu[pl] = *q[pl] = std::nan("");
      continue;
    }
    const double sinmu = std::copysign(std::sqrt(1.0 - cosmu * cosmu), m12);
    *bet[pl] = m12 / sinmu;
    *alf[pl] = (m11 - m22) / (2.0 * sinmu);
    *mu[pl] = std::atan2(sinmu, cosmu);
    double frac = *mu[pl] / (2.0 * 3.14159265358979323846);
    frac -= std::floor(frac);
    *q[pl] = frac;
  }
  *out = res;
  return done(XT_OK);
}

namespace xt {
namespace {
// The optics at delta0 and the closed orbits / tunes at delta0 -+ ddelta; dispersion and chromaticity from them.
int chromatic_twiss(const xt_lattice *lat, double delta0, double ddelta, const double *guess4,
                    xt_twiss4d_chrom_result &res, xt_twiss4d_result &hi, xt_twiss4d_result &lo, void *cuda_stream) {
  res = xt_twiss4d_chrom_result{};
  int rc = xt_twiss4d(lat, delta0, guess4, &res.on, cuda_stream);
  if (rc == XT_OK) rc = xt_twiss4d(lat, delta0 + ddelta, res.on.co, &hi, cuda_stream);
  if (rc == XT_OK) rc = xt_twiss4d(lat, delta0 - ddelta, res.on.co, &lo, cuda_stream);
  if (rc != XT_OK) return rc;
  double *d[4] = {&res.dx, &res.dpx, &res.dy, &res.dpy};
  for (int c = 0; c < 4; ++c) *d[c] = (hi.co[c] - lo.co[c]) / (2.0 * ddelta);
  auto slope = [&](double a, double b) {
    double diff = a - b;
    diff -= std::nearbyint(diff);  // fractional tunes live on a circle
    return diff / (2.0 * ddelta);  // NaN in, NaN out
  };
  res.dqx = slope(hi.qx_frac, lo.qx_frac);
  res.dqy = slope(hi.qy_frac, lo.qy_frac);
  return XT_OK;
}
}  // namespace
}  // namespace xt

static int xt_twiss4d_chrom_impl(const xt_lattice *lat, double delta0, double ddelta, const double *guess4,
                                xt_twiss4d_chrom_result *out, void *cuda_stream) {
  using namespace xt;
  if (!out || !(ddelta > 0.0) || !std::isfinite(ddelta)) {
    set_error("xt_twiss4d_chrom: NULL result or ddelta not > 0");
    return XT_ERR_INVALID_ARG;
  }
  xt_twiss4d_chrom_result res{};
  xt_twiss4d_result hi{}, lo{};
  const int rc = chromatic_twiss(lat, delta0, ddelta, guess4, res, hi, lo, cuda_stream);
  if (rc != XT_OK) return rc;
  *out = res;
  return XT_OK;
}

static int xt_twiss4d_normal_form_impl(const double *m, xt_twiss4d_modes *out) {
  using namespace xt;
  using cplx = std::complex<double>;
  if (!m || !out) {
    set_error("xt_twiss4d_normal_form: NULL argument");
    return XT_ERR_INVALID_ARG;
  }
  xt_twiss4d_modes res;
  const double nan = std::nan("");
  double *all[] = {&res.q1_frac, &res.q2_frac, &res.betx1, &res.alfx1, &res.bety1, &res.alfy1,
                   &res.betx2, &res.alfx2, &res.bety2, &res.alfy2};
  for (double *p : all) *p = nan;
  for (int k = 0; k < 8; ++k) res.v1[k] = res.v2[k] = nan;
  res.stable = 0;
  res.degenerate = 0;
  *out = res;
  double m2[16];
  for (int r = 0; r < 4; ++r)
    for (int c = 0; c < 4; ++c) {
      double s = 0.0;
      for (int k = 0; k < 4; ++k) s += m[4 * r + k] * m[4 * k + c];
      m2[4 * r + c] = s;
    }
  const double a = m[0] + m[5] + m[10] + m[15], t2 = m2[0] + m2[5] + m2[10] + m2[15];
  const double b = 0.5 * (a * a - t2);
  double disc = a * a - 4.0 * (b - 2.0);
  if (!std::isfinite(disc)) return XT_OK;
  if (std::fabs(disc) < 1e-7) {  // |cos mu_1 - cos mu_2| < 1.6e-4: below what a central-difference Jacobian resolves
    out->stable = (std::fabs(0.5 * a) < 4.0) ? 1 : 0;
    out->degenerate = 1;
    return XT_OK;
  }
  if (disc < 0.0) return XT_OK;  // complex u: a coupling (sum) resonance, unstable
  const double rt = std::sqrt(disc);
  const double u[2] = {0.5 * (a + rt), 0.5 * (a - rt)};
  if (!(std::fabs(u[0]) < 2.0) || !(std::fabs(u[1]) < 2.0)) return XT_OK;
  cplx v[2][4];
  double q[2];
  for (int k = 0; k < 2; ++k) {
    // A = (M^2 - u_other M + 1) w, w the unit vector that gives the longest A
    double best[4] = {0, 0, 0, 0}, best_n = -1.0;
    for (int j = 0; j < 4; ++j) {
      double col[4], n2 = 0.0;
      for (int r = 0; r < 4; ++r) {
        col[r] = m2[4 * r + j] - u[1 - k] * m[4 * r + j] + (r == j ? 1.0 : 0.0);
        n2 += col[r] * col[r];
      }
      if (n2 > best_n) {
        best_n = n2;
        for (int r = 0; r < 4; ++r) best[r] = col[r];
      }
    }
    const double c = 0.5 * u[k], sn = std::sqrt(1.0 - c * c);
    cplx lam(c, sn);
    for (int r = 0; r < 4; ++r) {
      double ma = 0.0;
      for (int j = 0; j < 4; ++j) ma += m[4 * r + j] * best[j];
      v[k][r] = ma - std::conj(lam) * best[r];
    }
    // v^H S v = 2i * norm
    double norm = 0.5 * (std::conj(v[k][0]) * v[k][1] - std::conj(v[k][1]) * v[k][0] + std::conj(v[k][2]) * v[k][3] -
                         std::conj(v[k][3]) * v[k][2]).imag();
    if (norm < 0.0) {
      for (int r = 0; r < 4; ++r) v[k][r] = std::conj(v[k][r]);
      lam = std::conj(lam);
      norm = -norm;
    }
    if (!(norm > 0.0)) return XT_OK;
    for (int r = 0; r < 4; ++r) v[k][r] /= std::sqrt(norm);
    double f = std::atan2(lam.imag(), lam.real()) / (2.0 * 3.14159265358979323846);
    q[k] = f - std::floor(f);
  }
  const int first = std::norm(v[0][0]) >= std::norm(v[1][0]) ? 0 : 1;
  for (int k = 0; k < 2; ++k) {
    const int src = k == 0 ? first : 1 - first;
    const cplx ref = v[src][k == 0 ? 0 : 2];
    const cplx ph = std::abs(ref) > 0.0 ? std::abs(ref) / ref : cplx(1.0, 0.0);
    cplx w[4];
    for (int r = 0; r < 4; ++r) w[r] = v[src][r] * ph;
    double *vec = k == 0 ? res.v1 : res.v2;
    for (int r = 0; r < 4; ++r) {
      vec[2 * r] = w[r].real();
      vec[2 * r + 1] = w[r].imag();
    }
    (k == 0 ? res.q1_frac : res.q2_frac) = q[src];
    (k == 0 ? res.betx1 : res.betx2) = std::norm(w[0]);
    (k == 0 ? res.alfx1 : res.alfx2) = -(std::conj(w[0]) * w[1]).real();
    (k == 0 ? res.bety1 : res.bety2) = std::norm(w[2]);
    (k == 0 ? res.alfy1 : res.alfy2) = -(std::conj(w[2]) * w[3]).real();
  }
  res.stable = 1;
  *out = res;
  return XT_OK;
}

static int xt_twiss4d_line_impl(const xt_lattice *lat, double delta0, double ddelta, const double *guess4,
                               xt_twiss4d_chrom_result *start, xt_twiss_row *rows, int64_t cap, void *cuda_stream) {
  using namespace xt;
  if (!lat || !rows || !(ddelta > 0.0) || !std::isfinite(ddelta) || !std::isfinite(delta0)) {
    set_error("xt_twiss4d_line: NULL lattice / rows, or ddelta not > 0");
    return XT_ERR_INVALID_ARG;
  }
  if (const int rc_dev = check_device(lat, "xt_twiss4d_line")) return rc_dev;
  Line line;
  if (!read_line(lat->packed_host, line)) {
    set_error("xt_twiss4d_line: the lattice holds no readable packed buffer");
    return XT_ERR_INVALID_ARG;
  }
  const int64_t n_el = static_cast<int64_t>(line.el.size());
  if (cap < n_el + 1) {
    set_error("xt_twiss4d_line: rows must hold n_elements + 1 entries");
    return XT_ERR_INVALID_ARG;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  // the optics at the start and the off-momentum closed orbits
  xt_twiss4d_chrom_result on{};
  xt_twiss4d_result hi{}, lo{};
  int rc = chromatic_twiss(lat, delta0, ddelta, guess4, on, hi, lo, cuda_stream);
  if (rc != XT_OK) return rc;
  if (!on.on.stable) {
    set_error("xt_twiss4d_line: a plane is unstable at the start of the line");
    return XT_ERR_UNSTABLE;
  }
  // the monitored line: a monitor record in front of every element and one behind the last
  Writer w(line);
  for (int64_t i = 0; i <= n_el; ++i) {
    const double row = static_cast<double>(i);
    w.put(kMonitorType, 0, &row, 1);
    if (i < n_el) w.put(line.el[i]);
  }
  const std::vector<unsigned char> &buf = w.finish();
  PackOpts po;
  po.allow_monitor = true;
  xt_lattice *mon = nullptr;
  if ((rc = create_lattice(buf.data(), buf.size(), po, &mon)) != XT_OK) return rc;

  constexpr int kN = 11;
  const size_t n_rows = static_cast<size_t>(n_el + 1);
  double *d_rows = nullptr, *d_f64 = nullptr;
  int64_t *d_i64 = nullptr;
  std::vector<double> h_rows(n_rows * kN * 6);
  auto done = [&](int code) {
    if (d_rows) cudaFree(d_rows);
    if (d_f64) cudaFree(d_f64);
    if (d_i64) cudaFree(d_i64);
    xt_lattice_destroy(mon);
    return code;
  };
#define XT_TRYL(call)                               \
  do {                                              \
    cudaError_t e__ = (call);                       \
    if (e__ != cudaSuccess) return done(xt::cuda_fail(e__, #call)); \
  } while (0)
  XT_TRYL(cudaMalloc(&d_rows, h_rows.size() * sizeof(double)));
  XT_TRYL(cudaMalloc(&d_f64, 10 * 16 * sizeof(double)));
  XT_TRYL(cudaMalloc(&d_i64, 3 * 16 * sizeof(int64_t)));
  XT_TRYL(cudaMemsetAsync(d_rows, 0xff, h_rows.size() * sizeof(double), st));  // NaN: a row a lost probe never wrote
  double h[10][16] = {};
  for (int k = 0; k < kN; ++k) {
    const double *z = k == 9 ? hi.co : k == 10 ? lo.co : on.on.co;
    for (int c = 0; c < 4; ++c) h[c][k] = z[c];
    h[5][k] = k == 9 ? delta0 + ddelta : k == 10 ? delta0 - ddelta : delta0;
  }
  for (int c = 0; c < 4; ++c) {
    h[c][1 + 2 * c] += kStep[c];
    h[c][2 + 2 * c] -= kStep[c];
  }
  int64_t hi64[3][16] = {};
  for (int k = 0; k < kN; ++k) hi64[1][k] = 1;  // state
  XT_TRYL(cudaMemcpyAsync(d_f64, h, sizeof(h), cudaMemcpyHostToDevice, st));
  XT_TRYL(cudaMemcpyAsync(d_i64, hi64, sizeof(hi64), cudaMemcpyHostToDevice, st));
  xt_particles p{};
  double **d[10] = {&p.x, &p.px, &p.y, &p.py, &p.zeta, &p.delta, &p.ptau, &p.rpp, &p.rvv, &p.s};
  for (int k = 0; k < 10; ++k) *d[k] = d_f64 + 16 * k;
  p.at_turn = d_i64;
  p.state = d_i64 + 16;
  p.at_element = d_i64 + 32;
  if ((rc = launch_init_derived(mon, p, kN, st)) != XT_OK) return done(rc);
  mon->d_monitor_rows = d_rows;  // `mon` is private to this call
  if ((rc = xt_track(mon, &p, kN, 1, st)) != XT_OK) return done(rc);
  XT_TRYL(cudaMemcpyAsync(h_rows.data(), d_rows, h_rows.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
  XT_TRYL(cudaStreamSynchronize(st));
#undef XT_TRYL

  xt_twiss4d_modes modes{};
  xt_twiss4d_normal_form(on.on.m, &modes);
  const bool have_modes = modes.stable && !modes.degenerate;
  double mode_mu[2] = {0.0, 0.0}, mode_raw[2] = {0.0, 0.0};
  const double two_pi = 2.0 * 3.14159265358979323846;
  const double b0[2] = {on.on.betx, on.on.bety}, a0[2] = {on.on.alfx, on.on.alfy};
  double mu_prev[2] = {0.0, 0.0}, raw_prev[2] = {0.0, 0.0};
  for (size_t i = 0; i < n_rows; ++i) {
    const double *r = h_rows.data() + i * kN * 6;
    for (int k = 0; k < kN * 6; ++k)
      if (!std::isfinite(r[k])) {
        set_error("xt_twiss4d_line: a probe particle was lost before element " + std::to_string(i));
        return done(XT_ERR_UNSTABLE);
      }
    xt_twiss_row &o = rows[i];
    o.s = i < static_cast<size_t>(n_el) ? lat->s_table_host[i] : lat->info.circumference;
    o.x = r[0];
    o.px = r[1];
    o.y = r[2];
    o.py = r[3];
    double jac[4][4];
    for (int row = 0; row < 4; ++row)
      for (int c = 0; c < 4; ++c)
        jac[row][c] = (r[(1 + 2 * c) * 6 + row] - r[(2 + 2 * c) * 6 + row]) / (2.0 * kStep[c]);
    double *bet[2] = {&o.betx, &o.bety}, *alf[2] = {&o.alfx, &o.alfy}, *mu[2] = {&o.mux, &o.muy};
    for (int pl = 0; pl < 2; ++pl) {
      const int q = 2 * pl;
      const double m11 = jac[q][q], m12 = jac[q][q + 1], m21 = jac[q + 1][q], m22 = jac[q + 1][q + 1];
      const double g0 = (1.0 + a0[pl] * a0[pl]) / b0[pl];
      *bet[pl] = m11 * m11 * b0[pl] - 2.0 * m11 * m12 * a0[pl] + m12 * m12 * g0;
      *alf[pl] = -m11 * m21 * b0[pl] + (m11 * m22 + m12 * m21) * a0[pl] - m12 * m22 * g0;
      double raw = std::atan2(m12, m11 * b0[pl] - m12 * a0[pl]);
      if (raw < 0.0) raw += two_pi;
      double step = raw - raw_prev[pl];             // the phase never runs backwards: unwrap
      if (step < -1e-6) step += two_pi;
      if (i == 0) step = 0.0;
      mu_prev[pl] += step;
      raw_prev[pl] = raw;
      *mu[pl] = mu_prev[pl];
    }
    o.betx1 = o.bety1 = o.betx2 = o.bety2 = o.mu1 = o.mu2 = std::nan("");
    if (have_modes) {  // steps 4-5: the eigenvectors carried by the tracked Jacobian
      for (int k = 0; k < 2; ++k) {
        const double *vec = k == 0 ? modes.v1 : modes.v2;
        std::complex<double> w[4];
        for (int row = 0; row < 4; ++row) {
          w[row] = 0.0;
          for (int c = 0; c < 4; ++c) w[row] += jac[row][c] * std::complex<double>(vec[2 * c], vec[2 * c + 1]);
        }
        (k == 0 ? o.betx1 : o.betx2) = std::norm(w[0]);
        (k == 0 ? o.bety1 : o.bety2) = std::norm(w[2]);
        const std::complex<double> own = w[k == 0 ? 0 : 2];
        double raw = std::atan2(own.imag(), own.real());
        if (raw < 0.0) raw += two_pi;
        double step = raw - mode_raw[k];
        if (step < -1e-6) step += two_pi;
        if (i == 0) step = 0.0;
        mode_mu[k] += step;
        mode_raw[k] = raw;
        (k == 0 ? o.mu1 : o.mu2) = mode_mu[k];
      }
    }
    double *dd[4] = {&o.dx, &o.dpx, &o.dy, &o.dpy};
    for (int c = 0; c < 4; ++c) *dd[c] = (r[9 * 6 + c] - r[10 * 6 + c]) / (2.0 * ddelta);
  }
  if (start) *start = on;
  return done(XT_OK);
}

namespace xt {
namespace {
constexpr int kProbe6 = 13;
constexpr double kStep6[6] = {1e-6, 1e-8, 1e-6, 1e-8, 1e-5, 1e-8};

// One launch: the orbit z and its twelve neighbours for one turn (x, px, y, py, zeta, delta).
int one_turn_and_jacobian6(const xt_lattice *lat, double *d_f64, int64_t *d_i64, const double z[6], double out[6],
                           double jac[36], cudaStream_t st) {
  double h[10][16] = {};
  for (int k = 0; k < kProbe6; ++k)
    for (int c = 0; c < 6; ++c) h[c][k] = z[c];
  for (int c = 0; c < 6; ++c) {
    h[c][1 + 2 * c] += kStep6[c];
    h[c][2 + 2 * c] -= kStep6[c];
  }
  int64_t hi64[3][16] = {};
  for (int k = 0; k < kProbe6; ++k) hi64[1][k] = 1;
  XT_CUDA(cudaMemcpyAsync(d_f64, h, sizeof(h), cudaMemcpyHostToDevice, st));
  XT_CUDA(cudaMemcpyAsync(d_i64, hi64, sizeof(hi64), cudaMemcpyHostToDevice, st));
  xt_particles p{};
  double **d[10] = {&p.x, &p.px, &p.y, &p.py, &p.zeta, &p.delta, &p.ptau, &p.rpp, &p.rvv, &p.s};
  for (int k = 0; k < 10; ++k) *d[k] = d_f64 + 16 * k;
  p.at_turn = d_i64;
  p.state = d_i64 + 16;
  p.at_element = d_i64 + 32;
  int rc = launch_init_derived(lat, p, kProbe6, st);
  if (rc != XT_OK) return rc;
  if ((rc = xt_track(lat, &p, kProbe6, 1, st)) != XT_OK) return rc;
  double r[6][16];
  int64_t state[16];
  XT_CUDA(cudaMemcpyAsync(r, d_f64, sizeof(r), cudaMemcpyDeviceToHost, st));
  XT_CUDA(cudaMemcpyAsync(state, d_i64 + 16, sizeof(state), cudaMemcpyDeviceToHost, st));
  XT_CUDA(cudaStreamSynchronize(st));
  for (int k = 0; k < kProbe6; ++k) {
    bool ok = state[k] == 1;
    for (int c = 0; c < 6; ++c) ok = ok && std::isfinite(r[c][k]);
    if (!ok) {
      set_error("xt_twiss6d: a probe particle was lost or became non-finite");
      return XT_ERR_UNSTABLE;
    }
  }
  for (int row = 0; row < 6; ++row) {
    out[row] = r[row][0];
    for (int c = 0; c < 6; ++c) jac[6 * row + c] = (r[row][1 + 2 * c] - r[row][2 + 2 * c]) / (2.0 * kStep6[c]);
  }
  return XT_OK;
}

int solve6(double a[6][7]) {  // Gaussian elimination with partial pivoting on [A | b]
  for (int c = 0; c < 6; ++c) {
    int piv = c;
    for (int r = c + 1; r < 6; ++r)
      if (std::fabs(a[r][c]) > std::fabs(a[piv][c])) piv = r;
    if (std::fabs(a[piv][c]) < 1e-300) return -1;
    if (piv != c)
      for (int k = 0; k < 7; ++k) std::swap(a[piv][k], a[c][k]);
    for (int r = c + 1; r < 6; ++r) {
      const double f = a[r][c] / a[c][c];
      for (int k = c; k < 7; ++k) a[r][k] -= f * a[c][k];
    }
  }
  for (int r = 5; r >= 0; --r) {
    double s = a[r][6];
    for (int k = r + 1; k < 6; ++k) s -= a[r][k] * a[k][6];
    a[r][6] = s / a[r][r];
  }
  return 0;
}
}  // namespace
}  // namespace xt

static int xt_twiss6d_impl(const xt_lattice *lat, const double *guess6, xt_twiss6d_result *out, void *cuda_stream) {
  using namespace xt;
  if (!lat || !out) {
    set_error("xt_twiss6d: NULL lattice or result");
    return XT_ERR_INVALID_ARG;
  }
  if (const int rc_dev = check_device(lat, "xt_twiss6d")) return rc_dev;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double *d_f64 = nullptr;
  int64_t *d_i64 = nullptr;
  XT_CUDA(cudaMalloc(&d_f64, 10 * 16 * sizeof(double)));
  cudaError_t e = cudaMalloc(&d_i64, 3 * 16 * sizeof(int64_t));
  if (e != cudaSuccess) {
    cudaFree(d_f64);
    return cuda_fail(e, "cudaMalloc(probe)");
  }
  auto done = [&](int code) {
    cudaFree(d_f64);
    cudaFree(d_i64);
    return code;
  };
  xt_twiss6d_result res{};
  double z[6] = {0, 0, 0, 0, 0, 0}, img[6], jac[36];
  if (guess6)
    for (int c = 0; c < 6; ++c) z[c] = guess6[c];
  int rc;
  bool converged = false;
  for (int it = 0; it < 25; ++it) {
    if ((rc = one_turn_and_jacobian6(lat, d_f64, d_i64, z, img, jac, st)) != XT_OK) return done(rc);
    double a[6][7];
    for (int r = 0; r < 6; ++r) {
      for (int c = 0; c < 6; ++c) a[r][c] = jac[6 * r + c] - (r == c ? 1.0 : 0.0);
      a[r][6] = -(img[r] - z[r]);
    }
    // without a cavity delta is invariant and zeta slips: the row of delta in M - 1 vanishes
    double row5 = 0.0;
    for (int c = 0; c < 6; ++c) row5 = std::fmax(row5, std::fabs(a[5][c]));
    if (row5 < 1e-12 || solve6(a) != 0) {
      set_error("xt_twiss6d: one-turn matrix minus identity is singular (no RF cavity, or an integer tune)");
      return done(XT_ERR_UNSTABLE);
    }
    double step = 0.0;
    for (int c = 0; c < 6; ++c) {
      z[c] += a[c][6];
      step = std::fmax(step, std::fabs(a[c][6]));
    }
    res.iterations = it + 1;
    if (step < 1e-12) {
      converged = true;
      break;
    }
  }
  if (!converged) {
    set_error("xt_twiss6d: closed-orbit search did not converge in 25 Newton steps");
    return done(XT_ERR_UNSTABLE);
  }
  if ((rc = one_turn_and_jacobian6(lat, d_f64, d_i64, z, img, jac, st)) != XT_OK) return done(rc);
  for (int c = 0; c < 6; ++c) res.co[c] = z[c];
  for (int k = 0; k < 36; ++k) res.m[k] = jac[k];
  // traces of M, M^2, M^3 -> elementary symmetric functions -> the cubic in u = lambda + 1/lambda
  double m2[36], m3[36];
  auto mul = [](const double *x, const double *y, double *o) {
    for (int r = 0; r < 6; ++r)
      for (int c = 0; c < 6; ++c) {
        double s = 0.0;
        for (int k = 0; k < 6; ++k) s += x[6 * r + k] * y[6 * k + c];
        o[6 * r + c] = s;
      }
  };
  mul(jac, jac, m2);
  mul(m2, jac, m3);
  double t1 = 0, t2 = 0, t3 = 0;
  for (int k = 0; k < 6; ++k) {
    t1 += jac[7 * k];
    t2 += m2[7 * k];
    t3 += m3[7 * k];
  }
  const double e1 = t1, e2 = 0.5 * (e1 * t1 - t2), e3 = (e2 * t1 - e1 * t2 + t3) / 3.0;
  const double s1 = e1, s2 = e2 - 3.0, s3 = e3 - 2.0 * e1;
  // u = w + s1/3: w^3 + p w + q = 0, three real roots by the trigonometric form
  const double pp = s2 - s1 * s1 / 3.0, qq = -2.0 * s1 * s1 * s1 / 27.0 + s1 * s2 / 3.0 - s3;
  double u[3];
  if (!(pp < 0.0)) {
    set_error("xt_twiss6d: the one-turn matrix has no three distinct stable modes");
    return done(XT_ERR_UNSTABLE);
  }
  const double amp = 2.0 * std::sqrt(-pp / 3.0);
  double arg = 3.0 * qq / (pp * amp);
  if (std::fabs(arg) > 1.0 + 1e-9) {
    set_error("xt_twiss6d: complex eigenvalue pair off the unit circle (unstable)");
    return done(XT_ERR_UNSTABLE);
  }
  arg = std::fmax(-1.0, std::fmin(1.0, arg));
  const double th = std::acos(arg) / 3.0;
  for (int k = 0; k < 3; ++k) u[k] = amp * std::cos(th - 2.0 * 3.14159265358979323846 * k / 3.0) + s1 / 3.0;
  double ang[3];
  for (int k = 0; k < 3; ++k) {
    if (!(std::fabs(u[k]) < 2.0)) {
      set_error("xt_twiss6d: an eigenvalue pair is off the unit circle (unstable)");
      return done(XT_ERR_UNSTABLE);
    }
    ang[k] = std::acos(0.5 * u[k]);
  }
  std::sort(ang, ang + 3);
  const double two_pi = 2.0 * 3.14159265358979323846;
  res.qs = ang[0] / two_pi;
  const double cx = 0.5 * (jac[0] + jac[7]);
  double a1 = ang[1], a2 = ang[2];
  if (std::fabs(std::cos(a1) - cx) > std::fabs(std::cos(a2) - cx)) std::swap(a1, a2);
  auto frac = [&](double a, double m12) {
    double f = std::copysign(a, m12) / two_pi;
    return f - std::floor(f);
  };
  res.q1_frac = frac(a1, jac[1]);
  res.q2_frac = frac(a2, jac[6 * 2 + 3]);
  *out = res;
  return done(XT_OK);
}

// C ABI: no C++ exception may cross it (include/xt.h: "No exceptions, no abort()").  The bodies above use
// std::vector / std::map / std::string; a failed host allocation comes back as XT_ERR_NOMEM.
extern "C" int xt_twiss4d(const xt_lattice *lat, double delta0, const double *guess4, xt_twiss4d_result *out, void *cuda_stream) {
  return xt::guarded<int>([&] { return xt_twiss4d_impl(lat, delta0, guess4, out, cuda_stream); });
}

extern "C" int xt_twiss4d_chrom(const xt_lattice *lat, double delta0, double ddelta, const double *guess4, xt_twiss4d_chrom_result *out, void *cuda_stream) {
  return xt::guarded<int>([&] { return xt_twiss4d_chrom_impl(lat, delta0, ddelta, guess4, out, cuda_stream); });
}

extern "C" int xt_twiss4d_line(const xt_lattice *lat, double delta0, double ddelta, const double *guess4, xt_twiss4d_chrom_result *start, xt_twiss_row *rows, int64_t cap, void *cuda_stream) {
  return xt::guarded<int>([&] { return xt_twiss4d_line_impl(lat, delta0, ddelta, guess4, start, rows, cap, cuda_stream); });
}

extern "C" int xt_twiss6d(const xt_lattice *lat, const double *guess6, xt_twiss6d_result *out, void *cuda_stream) {
  return xt::guarded<int>([&] { return xt_twiss6d_impl(lat, guess6, out, cuda_stream); });
}

extern "C" int xt_twiss4d_normal_form(const double *m, xt_twiss4d_modes *out) {
  return xt::guarded<int>([&] { return xt_twiss4d_normal_form_impl(m, out); });
}
