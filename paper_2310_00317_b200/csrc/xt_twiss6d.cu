// Twiss from tracking in six dimensions, steps 3-5: "the Linear Normal
// Form of the map [is obtained] from the eigenvalues and eigenvectors of the Jacobian matrix", the eigenvectors
// are propagated "to all other elements by tracking", and the Mais-Ripken functions and the dispersion follow
// from them.  xt_twiss6d (xt_twiss.cu) supplies the closed orbit and the 6x6 matrix; this file adds
//   xt_twiss6d_normal_form : host arithmetic on that matrix (no CUDA call),
//   xt_twiss6d_line        : one launch of thirteen probes through a monitored copy of the line, then the
//                            eigenvectors carried by the tracked Jacobians.
// The matrix of a symplectic map has a reciprocal characteristic polynomial: with u = lambda + 1/lambda the
// three pairs solve a cubic with real roots 2 cos mu_k (closed form, as in xt_twiss6d), and the eigenvector of
// exp(i mu_k) is (M - conj(lambda_k)) prod_{j != k} (M^2 - u_j M + 1) w for almost every w: no iterative
// eigen-solver.  The oracle procedure (oracle/make_optics.py: normal_form6, optics6d_along) uses
// numpy.linalg.eig instead.
#include <cmath>

#include <algorithm>
#include <complex>
#include <string>
#include <vector>

#include "xt_internal.h"
#include "xt_line.h"

namespace xt {
namespace {

using cplx = std::complex<double>;
constexpr double kTwoPi = 2.0 * 3.14159265358979323846;
constexpr int kProbe6 = 13;
constexpr double kStep6[6] = {1e-6, 1e-8, 1e-6, 1e-8, 1e-5, 1e-8};

void mul6(const double *x, const double *y, double *o) {
  for (int r = 0; r < 6; ++r)
    for (int c = 0; c < 6; ++c) {
      double s = 0.0;
      for (int k = 0; k < 6; ++k) s += x[6 * r + k] * y[6 * k + c];
      o[6 * r + c] = s;
    }
}

// Im(v^H S v)/2 for the block-diagonal S of (x, px), (y, py), (zeta, pzeta)
double symplectic_norm(const cplx v[6]) {
  double s = 0.0;
  for (int k = 0; k < 3; ++k) s += (std::conj(v[2 * k]) * v[2 * k + 1] - std::conj(v[2 * k + 1]) * v[2 * k]).imag();
  return 0.5 * s;
}

// delta -> rvv = beta/beta0 (the init helper's arithmetic)
double rvv_of_delta(double delta, double beta0) {
  const double ib = 1.0 / beta0;
  const double t = delta * (delta + 2.0);
  const double ptau = t / (std::sqrt(t + ib * ib) + ib);
  return (1.0 + delta) / (1.0 + beta0 * ptau);
}

void fill_nan(xt_twiss6d_modes &m) {
  const double nan = std::nan("");
  for (int k = 0; k < 3; ++k) {
    m.q_frac[k] = nan;
    for (int u = 0; u < 3; ++u) m.bet[u][k] = m.alf[u][k] = nan;
    for (int c = 0; c < 12; ++c) m.v[k][c] = nan;
  }
  for (int c = 0; c < 4; ++c) m.disp[c] = nan;
  m.stable = 0;
  m.degenerate = 0;
}

void functions_of(const cplx v[3][6], double rvv, double bet[3][3], double alf[3][3], double disp[4]) {
  for (int k = 0; k < 3; ++k)
    for (int u = 0; u < 3; ++u) {
      bet[u][k] = std::norm(v[k][2 * u]);
      alf[u][k] = -(std::conj(v[k][2 * u]) * v[k][2 * u + 1]).real();
    }
  for (int c = 0; c < 4; ++c) disp[c] = (v[2][c] / v[2][5]).real() * rvv;
}

}  // namespace
}  // namespace xt

static int xt_twiss6d_normal_form_impl(const double *m, double rvv_co, xt_twiss6d_modes *out) {
  using namespace xt;
  if (!m || !out || !(rvv_co > 0.0) || !std::isfinite(rvv_co)) {
    set_error("xt_twiss6d_normal_form: NULL argument or rvv_co not > 0");
    return XT_ERR_INVALID_ARG;
  }
  xt_twiss6d_modes res;
  fill_nan(res);
  *out = res;
  // canonical variables: pzeta = ptau/beta0, d pzeta = rvv d delta
  double jc[36];
  for (int r = 0; r < 6; ++r)
    for (int c = 0; c < 6; ++c) {
      double v = m[6 * r + c];
      if (r == 5) v *= rvv_co;
      if (c == 5) v /= rvv_co;
      jc[6 * r + c] = v;
      if (!std::isfinite(v)) return XT_OK;
    }
  double m2[36], m3[36];
  mul6(jc, jc, m2);
  mul6(m2, jc, m3);
  double t1 = 0, t2 = 0, t3 = 0;
  for (int k = 0; k < 6; ++k) {
    t1 += jc[7 * k];
    t2 += m2[7 * k];
    t3 += m3[7 * k];
  }
  const double e1 = t1, e2 = 0.5 * (e1 * t1 - t2), e3 = (e2 * t1 - e1 * t2 + t3) / 3.0;
  const double s1 = e1, s2 = e2 - 3.0, s3 = e3 - 2.0 * e1;
  const double pp = s2 - s1 * s1 / 3.0, qq = -2.0 * s1 * s1 * s1 / 27.0 + s1 * s2 / 3.0 - s3;
  if (!(pp < 0.0)) return XT_OK;
  const double amp = 2.0 * std::sqrt(-pp / 3.0);
  double arg = 3.0 * qq / (pp * amp);
  if (!(std::fabs(arg) <= 1.0 + 1e-9)) return XT_OK;  // a complex pair of u: off the unit circle
  arg = std::fmax(-1.0, std::fmin(1.0, arg));
  const double th = std::acos(arg) / 3.0;
  double u[3];
  for (int k = 0; k < 3; ++k) u[k] = amp * std::cos(th - kTwoPi * k / 3.0) + s1 / 3.0;
  for (int k = 0; k < 3; ++k)
    if (!(std::fabs(u[k]) < 2.0)) return XT_OK;
  res.stable = 1;
  for (int j = 0; j < 3; ++j)
    for (int k = j + 1; k < 3; ++k)
      if (std::fabs(u[j] - u[k]) < 3.2e-4) res.degenerate = 1;  // |cos mu_j - cos mu_k| < 1.6e-4 (see xt_twiss4d_normal_form)
  if (res.degenerate) {
    *out = res;
    return XT_OK;
  }
  cplx v[3][6];
  cplx lam[3];
  for (int k = 0; k < 3; ++k) {
    const double ua = u[(k + 1) % 3], ub = u[(k + 2) % 3];
    // B = (M^2 - ua M + 1)(M^2 - ub M + 1) = M^4 - (ua + ub) M^3 + (2 + ua ub) M^2 - (ua + ub) M + 1
    double m4[36], b[36];
    mul6(m2, m2, m4);
    for (int i = 0; i < 36; ++i)
      b[i] = m4[i] - (ua + ub) * m3[i] + (2.0 + ua * ub) * m2[i] - (ua + ub) * jc[i] + ((i % 7 == 0) ? 1.0 : 0.0);
    int best_j = 0;
    double best_n = -1.0;
    for (int j = 0; j < 6; ++j) {
      double n2 = 0.0;
      for (int r = 0; r < 6; ++r) n2 += b[6 * r + j] * b[6 * r + j];
      if (n2 > best_n) {
        best_n = n2;
        best_j = j;
      }
    }
    const double c = 0.5 * u[k], sn = std::sqrt(1.0 - c * c);
    lam[k] = cplx(c, sn);
    for (int r = 0; r < 6; ++r) {
      double ma = 0.0;
      for (int j = 0; j < 6; ++j) ma += jc[6 * r + j] * b[6 * j + best_j];
      v[k][r] = ma - std::conj(lam[k]) * b[6 * r + best_j];
    }
    double norm = symplectic_norm(v[k]);
    if (norm < 0.0) {
      for (int r = 0; r < 6; ++r) v[k][r] = std::conj(v[k][r]);
      lam[k] = std::conj(lam[k]);
      norm = -norm;
    }
    if (!(norm > 0.0)) {
      res.stable = 0;
      *out = res;
      return XT_OK;
    }
    for (int r = 0; r < 6; ++r) v[k][r] /= std::sqrt(norm);
  }
  // mode 3 = the smallest tune angle (longitudinal); of the other two, mode 1 has the larger horizontal part
  int order[3] = {0, 1, 2};
  std::sort(order, order + 3, [&](int a, int b2) { return std::fabs(std::arg(lam[a])) < std::fabs(std::arg(lam[b2])); });
  const int lon = order[0];
  int ta = order[1], tb = order[2];
  if (std::norm(v[tb][0]) > std::norm(v[ta][0])) std::swap(ta, tb);
  const int pick[3] = {ta, tb, lon};
  cplx w[3][6];
  for (int k = 0; k < 3; ++k) {
    const cplx ref = v[pick[k]][2 * k];
    const cplx ph = std::abs(ref) > 0.0 ? std::abs(ref) / ref : cplx(1.0, 0.0);
    for (int r = 0; r < 6; ++r) {
      w[k][r] = v[pick[k]][r] * ph;
      res.v[k][2 * r] = w[k][r].real();
      res.v[k][2 * r + 1] = w[k][r].imag();
    }
    const double f = std::arg(lam[pick[k]]) / kTwoPi;
    res.q_frac[k] = f - std::floor(f);
  }
  functions_of(w, rvv_co, res.bet, res.alf, res.disp);
  *out = res;
  return XT_OK;
}

static int xt_twiss6d_line_impl(const xt_lattice *lat, const double *guess6, xt_twiss6d_result *start,
                                xt_twiss6d_modes *start_modes, xt_twiss6d_row *rows, int64_t cap, void *cuda_stream) {
  using namespace xt;
  if (!lat || !rows) {
    set_error("xt_twiss6d_line: NULL lattice or rows");
    return XT_ERR_INVALID_ARG;
  }
  if (const int rc_dev = check_device(lat, "xt_twiss6d_line")) return rc_dev;
  Line line;
  if (!read_line(lat->packed_host, line)) {
    set_error("xt_twiss6d_line: the lattice holds no readable packed buffer");
    return XT_ERR_INVALID_ARG;
  }
  const int64_t n_el = static_cast<int64_t>(line.el.size());
  if (cap < n_el + 1) {
    set_error("xt_twiss6d_line: rows must hold n_elements + 1 entries");
    return XT_ERR_INVALID_ARG;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  xt_twiss6d_result on{};
  int rc = xt_twiss6d(lat, guess6, &on, cuda_stream);
  if (rc != XT_OK) return rc;
  const double beta0 = lat->k.beta0;
  const double rvv0 = rvv_of_delta(on.co[5], beta0);
  xt_twiss6d_modes modes{};
  if ((rc = xt_twiss6d_normal_form(on.m, rvv0, &modes)) != XT_OK) return rc;
  if (!modes.stable || modes.degenerate) {
    set_error("xt_twiss6d_line: the one-turn matrix has no three distinct stable modes");
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
  const size_t n_rows = static_cast<size_t>(n_el + 1);
  double *d_rows = nullptr, *d_f64 = nullptr;
  int64_t *d_i64 = nullptr;
  std::vector<double> h_rows(n_rows * kProbe6 * 6);
  auto done = [&](int code) {
    if (d_rows) cudaFree(d_rows);
    if (d_f64) cudaFree(d_f64);
    if (d_i64) cudaFree(d_i64);
    xt_lattice_destroy(mon);
    return code;
  };
#define XT_TRYL(call)                                               \
  do {                                                              \
    cudaError_t e__ = (call);                                       \
    if (e__ != cudaSuccess) return done(xt::cuda_fail(e__, #call)); \
  } while (0)
  XT_TRYL(cudaMalloc(&d_rows, h_rows.size() * sizeof(double)));
  XT_TRYL(cudaMalloc(&d_f64, 10 * 16 * sizeof(double)));
  XT_TRYL(cudaMalloc(&d_i64, 3 * 16 * sizeof(int64_t)));
  XT_TRYL(cudaMemsetAsync(d_rows, 0xff, h_rows.size() * sizeof(double), st));  // NaN: a row a lost probe never wrote
  double h[10][16] = {};
  for (int k = 0; k < kProbe6; ++k)
    for (int c = 0; c < 6; ++c) h[c][k] = on.co[c];
  for (int c = 0; c < 6; ++c) {
    h[c][1 + 2 * c] += kStep6[c];
    h[c][2 + 2 * c] -= kStep6[c];
  }
  int64_t hi64[3][16] = {};
  for (int k = 0; k < kProbe6; ++k) hi64[1][k] = 1;  // state
  XT_TRYL(cudaMemcpyAsync(d_f64, h, sizeof(h), cudaMemcpyHostToDevice, st));
  XT_TRYL(cudaMemcpyAsync(d_i64, hi64, sizeof(hi64), cudaMemcpyHostToDevice, st));
  xt_particles p{};
  double **d[10] = {&p.x, &p.px, &p.y, &p.py, &p.zeta, &p.delta, &p.ptau, &p.rpp, &p.rvv, &p.s};
  for (int k = 0; k < 10; ++k) *d[k] = d_f64 + 16 * k;
  p.at_turn = d_i64;
  p.state = d_i64 + 16;
  p.at_element = d_i64 + 32;
  if ((rc = launch_init_derived(mon, p, kProbe6, st)) != XT_OK) return done(rc);
  mon->d_monitor_rows = d_rows;  // `mon` is private to this call
  if ((rc = xt_track(mon, &p, kProbe6, 1, st)) != XT_OK) return done(rc);
  XT_TRYL(cudaMemcpyAsync(h_rows.data(), d_rows, h_rows.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
  XT_TRYL(cudaStreamSynchronize(st));
#undef XT_TRYL

  cplx v0[3][6];
  for (int k = 0; k < 3; ++k)
    for (int r = 0; r < 6; ++r) v0[k][r] = cplx(modes.v[k][2 * r], modes.v[k][2 * r + 1]);
  double mu_acc[3] = {0, 0, 0}, raw_prev[3] = {0, 0, 0};
  for (size_t i = 0; i < n_rows; ++i) {
    const double *r = h_rows.data() + i * kProbe6 * 6;
    for (int k = 0; k < kProbe6 * 6; ++k)
      if (!std::isfinite(r[k])) {
        set_error("xt_twiss6d_line: a probe particle was lost before element " + std::to_string(i));
        return done(XT_ERR_UNSTABLE);
      }
    xt_twiss6d_row &o = rows[i];
    o.s = i < static_cast<size_t>(n_el) ? lat->s_table_host[i] : lat->info.circumference;
    for (int c = 0; c < 6; ++c) o.co[c] = r[c];
    const double rvv1 = rvv_of_delta(r[5], beta0);
    // Jacobian from the start to this row in canonical variables at both ends
    double jac[6][6];
    for (int row = 0; row < 6; ++row)
      for (int c = 0; c < 6; ++c) {
        double v = (r[(1 + 2 * c) * 6 + row] - r[(2 + 2 * c) * 6 + row]) / (2.0 * kStep6[c]);
        if (row == 5) v *= rvv1;
        if (c == 5) v /= rvv0;
        jac[row][c] = v;
      }
    cplx wv[3][6];
    for (int k = 0; k < 3; ++k)
      for (int row = 0; row < 6; ++row) {
        wv[k][row] = 0.0;
        for (int c = 0; c < 6; ++c) wv[k][row] += jac[row][c] * v0[k][c];
      }
    functions_of(wv, rvv1, o.bet, o.alf, o.disp);
    for (int k = 0; k < 3; ++k) {
      // phase of the mode's own component, unwrapped along the line.  A betatron phase only grows; the slow
      // synchrotron phase runs backwards above transition (q_frac[2] just below 1): it is counted in its own sense
      const cplx own = wv[k][2 * k];
      double raw = std::atan2(own.imag(), own.real());
      const double sense = (k == 2 && modes.q_frac[2] > 0.5) ? -1.0 : 1.0;
      double step = sense * (raw - raw_prev[k]);
      while (step < -1e-6) step += kTwoPi;
      while (step >= kTwoPi - 1e-6) step -= kTwoPi;
      if (i == 0) step = 0.0;
      mu_acc[k] += step;
      raw_prev[k] = raw;
      o.mu[k] = mu_acc[k];
    }
  }
  if (start) *start = on;
  if (start_modes) *start_modes = modes;
  return done(XT_OK);
}

extern "C" int xt_twiss6d_normal_form(const double *m, double rvv_co, xt_twiss6d_modes *out) {
  return xt::guarded<int>([&] { return xt_twiss6d_normal_form_impl(m, rvv_co, out); });
}

extern "C" int xt_twiss6d_line(const xt_lattice *lat, const double *guess6, xt_twiss6d_result *start,
                               xt_twiss6d_modes *start_modes, xt_twiss6d_row *rows, int64_t cap, void *cuda_stream) {
  return xt::guarded<int>([&] { return xt_twiss6d_line_impl(lat, guess6, start, start_modes, rows, cap, cuda_stream); });
}
