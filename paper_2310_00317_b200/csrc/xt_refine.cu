// Loss-location refinement ("particle backtracking and a locally
// refined aperture model obtained by polygonal interpolation", Fig. 4; DESIGN.md reading
// A20, section 16).
//
// Host side: geometry only -- the frame (accumulated XYShift / SRotation) in front of every element, the
// two apertures sampled on n_poly rays, and, per flagging aperture, two small packed lattices: the
// elements back to the upstream aperture in reverse order (reading A11: reversed line + sign flips =
// inverse map), and the same elements forward with every length cut into pieces of at most ds, a
// polygon aperture after each piece.  Device side: gather the lost particles of that aperture into a
// compact ensemble (flipping px, py, zeta), xt_track it through the first lattice, flip again, xt_track
// it through the second, scatter the records the polygons stopped back into the caller's arrays.
// Every map runs in the tracking kernels of xt_track.cu; nothing is tracked on the host.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>
#include <string>
#include <vector>

#include "xt_internal.h"
#include "xt_line.h"

namespace xt {
namespace {

// Frame in front of an element: local = R m + t, R = [[c, s], [-s, c]] (tilts and
// misalignments are changes of the reference system).
struct Frame {
  double c = 1.0, s = 0.0, tx = 0.0, ty = 0.0;
};

std::vector<Frame> frames_of(const Line &line) {
  std::vector<Frame> out(line.el.size() + 1);
  Frame f;
  for (size_t i = 0; i < line.el.size(); ++i) {
    out[i] = f;
    const Elem &e = line.el[i];
    if (e.type == XT_XYSHIFT) {
      f.tx -= e.v[0];
      f.ty -= e.v[1];
    } else if (e.type == XT_SROTATION) {
      const double cz = e.v[0], sz = e.v[1];
      const Frame g = f;
      f.c = cz * g.c - sz * g.s;
      f.s = cz * g.s + sz * g.c;
      f.tx = cz * g.tx + sz * g.ty;
      f.ty = cz * g.ty - sz * g.tx;
    }
  }
  out[line.el.size()] = f;
  return out;
}

// One LimitRect / LimitEllipse / LimitPolygon sampled on n rays from its centre at machine-frame angles
// 2 pi k / n.  false: a polygon that does not surround the mean of its vertices.
bool sample_aperture(const Elem &e, const Frame &f, int n, std::vector<double> &vx, std::vector<double> &vy) {
  const double pi = 3.14159265358979323846264338327950288;
  double cx = 0.0, cy = 0.0, hx = 0.0, hy = 0.0;
  if (e.type == XT_LIMITRECT) {
    cx = 0.5 * (e.v[0] + e.v[1]);
    cy = 0.5 * (e.v[2] + e.v[3]);
    hx = 0.5 * (e.v[1] - e.v[0]);
    hy = 0.5 * (e.v[3] - e.v[2]);
  }
  const int nv = e.type == XT_LIMITPOLYGON ? static_cast<int>(e.aux) : 0;
  if (nv) {  // centre: the mean of the vertices (x[0..nv), y[0..nv))
    for (int i = 0; i < nv; ++i) {
      cx += e.v[i];
      cy += e.v[nv + i];
    }
    cx /= nv;
    cy /= nv;
  }
  const double lx = cx - f.tx, ly = cy - f.ty;  // centre in the machine frame: R^T (local - t)
  const double mx = f.c * lx - f.s * ly, my = f.s * lx + f.c * ly;
  vx.resize(n);
  vy.resize(n);
  for (int k = 0; k < n; ++k) {
    const double phi = (2.0 * pi * k) / n;
    const double dx = std::cos(phi), dy = std::sin(phi);
    const double ux = f.c * dx + f.s * dy, uy = f.c * dy - f.s * dx;  // the ray in the aperture's frame
    double r;
    if (e.type == XT_LIMITRECT) {
      const double rx = ux != 0.0 ? hx / std::fabs(ux) : INFINITY;
      const double ry = uy != 0.0 ? hy / std::fabs(uy) : INFINITY;
      r = std::fmin(rx, ry);
    } else if (nv) {
      // the ray c + r u meets the edge a + t (b - a): r = cross(a - c, e)/cross(u, e), t = cross(a - c, u)/cross(u, e)
      r = INFINITY;
      for (int i = 0; i < nv; ++i) {
        const int j = (i + 1) % nv;
        const double ax = e.v[i] - cx, ay = e.v[nv + i] - cy;
        const double ex = e.v[j] - e.v[i], ey = e.v[nv + j] - e.v[nv + i];
        const double den = ux * ey - uy * ex;
        if (den == 0.0) continue;
        const double rr = (ax * ey - ay * ex) / den, t = (ax * uy - ay * ux) / den;
        if (rr > 0.0 && t >= 0.0 && t <= 1.0 && rr < r) r = rr;
      }
      if (!std::isfinite(r)) return false;
    } else {
      const double qa = ux / e.v[0], qb = uy / e.v[1];
      r = 1.0 / std::sqrt(qa * qa + qb * qb);
    }
    vx[k] = mx + r * dx;
    vy[k] = my + r * dy;
  }
  return true;
}

struct Work {  // compact ensemble of one group, device
  double *f64 = nullptr;   // 10 arrays of cap doubles
  int64_t *i64 = nullptr;  // 3 arrays of cap int64 + cap indices
  int64_t cap = 0;
  xt_particles view() const {
    xt_particles p{};
    double **d[10] = {&p.x, &p.px, &p.y, &p.py, &p.zeta, &p.delta, &p.ptau, &p.rpp, &p.rvv, &p.s};
    for (int k = 0; k < 10; ++k) *d[k] = f64 + k * cap;
    p.at_turn = i64;
    p.state = i64 + cap;
    p.at_element = i64 + 2 * cap;
    p.particle_id = nullptr;
    return p;
  }
  int64_t *idx() const { return i64 + 3 * cap; }
};

__global__ void gather_kernel(xt_particles src, xt_particles dst, const int64_t *idx, int64_t n) {
  const int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
  if (i >= n) return;
  const int64_t k = idx[i];
  dst.x[i] = src.x[k];
  dst.px[i] = -src.px[k];  // reading A11: R = (x, -px, y, -py, -zeta, delta)
  dst.y[i] = src.y[k];
  dst.py[i] = -src.py[k];
  dst.zeta[i] = -src.zeta[k];
  dst.delta[i] = src.delta[k];
  dst.ptau[i] = src.ptau[k];
  dst.rpp[i] = src.rpp[k];
  dst.rvv[i] = src.rvv[k];
  dst.s[i] = 0.0;
  dst.at_turn[i] = 0;
  dst.state[i] = 1;
  dst.at_element[i] = 0;
}

__global__ void flip_kernel(xt_particles p, int64_t n) {
  const int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
  if (i >= n) return;
  p.px[i] = -p.px[i];
  p.py[i] = -p.py[i];
  p.zeta[i] = -p.zeta[i];
  p.at_turn[i] = 0;
  p.s[i] = 0.0;
}

__global__ void scatter_kernel(xt_particles src, xt_particles dst, const int64_t *idx, int64_t n, double s_u,
                               unsigned long long *moved) {
  const int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
  if (i >= n || src.state[i] != 0) return;  // passed every polygon: the record stays
  const int64_t k = idx[i];
  dst.x[k] = src.x[i];
  dst.px[k] = src.px[i];
  dst.y[k] = src.y[i];
  dst.py[k] = src.py[i];
  dst.zeta[k] = src.zeta[i];
  dst.delta[k] = src.delta[i];
  dst.ptau[k] = src.ptau[i];
  dst.rpp[k] = src.rpp[i];
  dst.rvv[k] = src.rvv[i];
  dst.s[k] = s_u + src.s[i];
  atomicAdd(moved, 1ull);
}

struct LatticeGuard {
  xt_lattice *lat = nullptr;
  ~LatticeGuard() { xt_lattice_destroy(lat); }
};

}  // namespace
}  // namespace xt

static int xt_refine_loss_location_impl(const xt_lattice *lat, const xt_particles *p, int64_t n_part, double ds,
                                       int32_t n_poly, int64_t *n_refined, void *cuda_stream) {
  using namespace xt;
  if (n_refined) *n_refined = 0;
  if (!lat || !p) {
    set_error("xt_refine_loss_location: lat or p is NULL");
    return XT_ERR_INVALID_ARG;
  }
  if (!(ds > 0.0) || !std::isfinite(ds) || n_poly < 3 || n_poly > 256 || n_part < 0) {
    set_error("xt_refine_loss_location: needs ds > 0, 3 <= n_poly <= 256, n_part >= 0");
    return XT_ERR_INVALID_ARG;
  }
  if (!p->x || !p->px || !p->y || !p->py || !p->zeta || !p->delta || !p->ptau || !p->rpp || !p->rvv || !p->s ||
      !p->at_turn || !p->state || !p->at_element) {
    set_error("xt_refine_loss_location: every particle array except particle_id is needed (at_element too)");
    return XT_ERR_INVALID_ARG;
  }
  if (n_part == 0) return XT_OK;
  const int rc_dev = check_device(lat, "xt_refine_loss_location");  // before any allocation or launch
  if (rc_dev != XT_OK) return rc_dev;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  Line line;
  if (!read_line(lat->packed_host, line)) {
    set_error("xt_refine_loss_location: the lattice holds no readable packed buffer");
    return XT_ERR_INVALID_ARG;
  }
  const std::vector<double> &s_tab = lat->s_table_host;
  const int64_t n_el = static_cast<int64_t>(line.el.size());

  // which particles, grouped by the aperture that flagged them
  std::vector<int64_t> state(n_part), at_el(n_part);
  XT_CUDA(cudaMemcpyAsync(state.data(), p->state, n_part * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  XT_CUDA(cudaMemcpyAsync(at_el.data(), p->at_element, n_part * sizeof(int64_t), cudaMemcpyDeviceToHost, st));
  XT_CUDA(cudaStreamSynchronize(st));
  std::vector<int64_t> lost;
  for (int64_t i = 0; i < n_part; ++i)
    if (state[i] == 0 && at_el[i] >= 0 && at_el[i] < n_el && line.el[at_el[i]].is_aperture()) lost.push_back(i);
  if (lost.empty()) return XT_OK;
  std::stable_sort(lost.begin(), lost.end(), [&](int64_t a, int64_t b) { return at_el[a] < at_el[b]; });
  int64_t cap = 0;
  for (size_t lo = 0; lo < lost.size();) {
    size_t hi = lo;
    while (hi < lost.size() && at_el[lost[hi]] == at_el[lost[lo]]) ++hi;
    cap = std::max<int64_t>(cap, static_cast<int64_t>(hi - lo));
    lo = hi;
  }

  Work w;
  w.cap = cap;
  unsigned long long *d_moved = nullptr;
  auto release = [&]() {
    if (w.f64) cudaFree(w.f64);
    if (w.i64) cudaFree(w.i64);
    if (d_moved) cudaFree(d_moved);
  };
#define XT_TRY(call)                      \
  do {                                    \
    cudaError_t e__ = (call);             \
    if (e__ != cudaSuccess) {             \
      release();                          \
      return xt::cuda_fail(e__, #call);   \
    }                                     \
  } while (0)
#define XT_TRY_RC(call)   \
  do {                    \
    const int rc__ = (call); \
    if (rc__ != XT_OK) {  \
      release();          \
      return rc__;        \
    }                     \
  } while (0)
  XT_TRY(cudaMalloc(&w.f64, 10 * cap * sizeof(double)));
  XT_TRY(cudaMalloc(&w.i64, 4 * cap * sizeof(int64_t)));
  XT_TRY(cudaMalloc(&d_moved, sizeof(unsigned long long)));
  XT_TRY(cudaMemsetAsync(d_moved, 0, sizeof(unsigned long long), st));
  const xt_particles tmp = w.view();
  const std::vector<Frame> frames = frames_of(line);

  std::vector<double> ux, uy, lx, ly, px(n_poly), py(n_poly), pv(2 * static_cast<size_t>(n_poly));
  for (size_t lo = 0; lo < lost.size();) {
    size_t hi = lo;
    const int64_t l = at_el[lost[lo]];
    while (hi < lost.size() && at_el[lost[hi]] == l) ++hi;
    const int64_t n_g = static_cast<int64_t>(hi - lo);
    const size_t g_lo = lo;
    lo = hi;
    int64_t u = l - 1;
    while (u >= 0 && !line.el[u].is_aperture()) --u;
    const double s_u = u >= 0 ? s_tab[u] : 0.0;
    const double seg_len = s_tab[l] - s_u;
    if (!(seg_len > 0.0)) continue;
    bool ok = sample_aperture(line.el[l], frames[l], n_poly, lx, ly);
    if (u >= 0) {
      ok = ok && sample_aperture(line.el[u], frames[u], n_poly, ux, uy);
    } else {
      ux = lx;
      uy = ly;
    }
    if (!ok) {
      release();
      set_error("xt_refine_loss_location: a polygon aperture does not surround the mean of its vertices");
      return XT_ERR_BAD_LATTICE;
    }

    // back: elements l-1 .. u+1, reversed (reading A11)
    Writer back(line);
    for (int64_t i = l - 1; i > u; --i) {
      Elem e = line.el[i];
      if (e.is_any_aperture()) continue;
      if (e.type == XT_CAVITY) e.v[2] = -e.v[2];
      if (e.type == XT_SROTATION) e.v[1] = -e.v[1];
      if (e.type == XT_XYSHIFT) {
        e.v[0] = -e.v[0];
        e.v[1] = -e.v[1];
      }
      back.put(e);
    }
    // forward: the same elements, lengths cut into pieces of at most ds, a polygon behind each piece
    Writer fine(line);
    double sloc = 0.0;
    for (int64_t i = u + 1; i < l; ++i) {
      const Elem &e = line.el[i];
      if (e.is_any_aperture()) continue;
      const double length = e.length();
      if (!(length > 0.0)) {
        fine.put(e);
        continue;
      }
      const int64_t n = static_cast<int64_t>(std::ceil(length / ds));
      const double piece = length / static_cast<double>(n);
      Elem cut = e;
      cut.v[e.type == XT_DRIFT ? 0 : e.type == XT_QUADRUPOLE ? 1 : 2] = piece;
      const Frame &f = frames[i];
      for (int64_t j = 0; j < n; ++j) {
        fine.put(cut);
        sloc = sloc + piece;
        const double lam = sloc / seg_len;
        for (int k = 0; k < n_poly; ++k) {
          const double mx = ux[k] + lam * (lx[k] - ux[k]);
          const double my = uy[k] + lam * (ly[k] - uy[k]);
          pv[k] = f.c * mx + f.s * my + f.tx;
          pv[n_poly + k] = f.c * my - f.s * mx + f.ty;
        }
        fine.put(XT_LIMITPOLYGON, static_cast<uint32_t>(n_poly), pv.data(), pv.size());
      }
    }

    LatticeGuard lb, lf;
    const std::vector<unsigned char> &bb = back.finish(), &fb = fine.finish();
    XT_TRY_RC(xt_lattice_create(bb.data(), bb.size(), &lb.lat));
    XT_TRY_RC(xt_lattice_create(fb.data(), fb.size(), &lf.lat));
    XT_TRY(cudaMemcpyAsync(w.idx(), lost.data() + g_lo, n_g * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    const int block = 128;
    const unsigned grid = static_cast<unsigned>((n_g + block - 1) / block);
    gather_kernel<<<grid, block, 0, st>>>(*p, tmp, w.idx(), n_g);
    XT_TRY(cudaGetLastError());
    XT_TRY_RC(xt_track(lb.lat, &tmp, n_g, 1, st));
    flip_kernel<<<grid, block, 0, st>>>(tmp, n_g);
    XT_TRY(cudaGetLastError());
    XT_TRY_RC(xt_track(lf.lat, &tmp, n_g, 1, st));
    scatter_kernel<<<grid, block, 0, st>>>(tmp, *p, w.idx(), n_g, s_u, d_moved);
    XT_TRY(cudaGetLastError());
    count_launch(3);
    XT_TRY(cudaStreamSynchronize(st));  // the lattices and the index staging die with this iteration
  }
  unsigned long long moved = 0;
  XT_TRY(cudaMemcpyAsync(&moved, d_moved, sizeof(moved), cudaMemcpyDeviceToHost, st));
  XT_TRY(cudaStreamSynchronize(st));
  release();
#undef XT_TRY
#undef XT_TRY_RC
  if (n_refined) *n_refined = static_cast<int64_t>(moved);
  return XT_OK;
}

// C ABI: no C++ exception may cross it (include/xt.h: "No exceptions, no abort()").  The bodies above use
// std::vector / std::map / std::string; a failed host allocation comes back as XT_ERR_NOMEM.
extern "C" int xt_refine_loss_location(const xt_lattice *lat, const xt_particles *p, int64_t n_part, double ds, int32_t n_poly, int64_t *n_refined, void *cuda_stream) {
  return xt::guarded<int>([&] { return xt_refine_loss_location_impl(lat, p, n_part, ds, n_poly, n_refined, cuda_stream); });
}
