// Time functions ("time dependent knobs that are updated automatically
// during the simulation", Fig. 1; reading A21, section 17).
//
// The lattice image stays what the tracking kernel streams; what changes with time is a handful of multipole
// coefficients in it.  xt_lattice_set_knobs resolves every link to the image offset of its coefficient (the
// packer records where each multipole's coefficient pairs went, fused or not) and keeps table, targets and
// links on the device.  xt_track_knobs then alternates, on one stream, a tiny kernel that rewrites those
// coefficients for the turn's step with the tracking kernel for one turn: no host round trip, no repacking,
// and the hot kernel is untouched.
#include <algorithm>
#include <cmath>
#include <map>
#include <tuple>
#include <vector>

#include "xt_internal.h"
#include "xt_line.h"

namespace xt {
namespace {

struct KnobTarget {
  uint64_t off;      // image offset of the coefficient (c[n] or s[n])
  uint64_t wf_off;   // image offset of the weak-focusing term that follows knl[0] of a curved multipole, or ~0
  double base;       // knl[n] / ksl[n] of the packed buffer
  double fact;       // n!
  double hxl;        // != 0: the normal dipole term of a curved multipole, stored as knl[0] - hxl
  double length;     // for the weak-focusing term (knl[0] hxl)/length
  int32_t first, count;  // its links
};
struct KnobLink {
  int32_t knob, pad;
  double gain;
};

// One thread per linked coefficient: the packer's arithmetic (xt_lattice.cu, XT_MULTIPOLE) on the knob value.
__global__ void apply_knobs_kernel(unsigned char *image, const KnobTarget *targets, const KnobLink *links,
                                   const double *table, int64_t n_steps, int64_t step, int64_t n_targets,
                                   int with_links) {
  const int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
  if (i >= n_targets) return;
  const KnobTarget t = targets[i];
  double v = t.base;
  if (with_links)
    for (int32_t k = 0; k < t.count; ++k) {
      const KnobLink l = links[t.first + k];
      v = __dadd_rn(v, __dmul_rn(l.gain, table[static_cast<int64_t>(l.knob) * n_steps + step]));
    }
  const double c = (t.hxl != 0.0) ? __dsub_rn(v, t.hxl) : __ddiv_rn(v, t.fact);
  *reinterpret_cast<double *>(image + t.off) = c;
  if (t.wf_off != ~0ull) *reinterpret_cast<double *>(image + t.wf_off) = __ddiv_rn(__dmul_rn(v, t.hxl), t.length);
}

void drop_knobs(xt_lattice *lat) {
  if (lat->d_knob_table) cudaFree(lat->d_knob_table);
  if (lat->d_knob_targets) cudaFree(lat->d_knob_targets);
  if (lat->d_knob_links) cudaFree(lat->d_knob_links);
  lat->d_knob_table = nullptr;
  lat->d_knob_targets = lat->d_knob_links = nullptr;
  lat->n_knob_targets = lat->n_knob_steps = 0;
}

int launch_apply(const xt_lattice *lat, int64_t step, int with_links, cudaStream_t st) {
  const int block = 128;
  const unsigned grid = static_cast<unsigned>((lat->n_knob_targets + block - 1) / block);
  apply_knobs_kernel<<<grid, block, 0, st>>>(lat->d_image, static_cast<const KnobTarget *>(lat->d_knob_targets),
                                             static_cast<const KnobLink *>(lat->d_knob_links), lat->d_knob_table,
                                             lat->n_knob_steps, step, lat->n_knob_targets, with_links);
  XT_CUDA(cudaGetLastError());
  count_launch(1);
  return XT_OK;
}

}  // namespace
}  // namespace xt

static int xt_lattice_set_knobs_impl(xt_lattice *lat, const double *table, int32_t n_knobs, int64_t n_steps,
                                    const xt_knob_link *links, int64_t n_links) {
  using namespace xt;
  if (!lat || n_links < 0) {
    set_error("xt_lattice_set_knobs: lat is NULL or n_links < 0");
    return XT_ERR_INVALID_ARG;
  }
  int rc_dev = check_device(lat, "xt_lattice_set_knobs");
  if (rc_dev != XT_OK) return rc_dev;
  if (n_links == 0) {
    drop_knobs(lat);
    return XT_OK;
  }
  if (!table || !links || n_knobs < 1 || n_steps < 1) {
    set_error("xt_lattice_set_knobs: needs a table of n_knobs >= 1 rows and n_steps >= 1 columns, and links");
    return XT_ERR_INVALID_ARG;
  }
  for (int64_t i = 0; i < static_cast<int64_t>(n_knobs) * n_steps; ++i)
    if (!std::isfinite(table[i])) {
      set_error("xt_lattice_set_knobs: non-finite knob value");
      return XT_ERR_INVALID_ARG;
    }
  Line line;
  if (!read_line(lat->packed_host, line)) {
    set_error("xt_lattice_set_knobs: the lattice holds no readable packed buffer");
    return XT_ERR_INVALID_ARG;
  }
  const int64_t n_el = static_cast<int64_t>(line.el.size());
  // group the links by coefficient, keeping the order in which they were given
  std::map<std::tuple<int64_t, int32_t, int32_t>, std::vector<KnobLink>> by_target;
  std::vector<std::tuple<int64_t, int32_t, int32_t>> order_seen;
  for (int64_t i = 0; i < n_links; ++i) {
    const xt_knob_link &l = links[i];
    if (l.element < 0 || l.element >= n_el || line.el[l.element].type != XT_MULTIPOLE || l.order < 0 ||
        l.order > static_cast<int32_t>(line.el[l.element].aux) || (l.skew != 0 && l.skew != 1) || l.knob < 0 ||
        l.knob >= n_knobs || !std::isfinite(l.gain) || lat->mult_slot0[l.element] == ~0ull) {
      set_error("xt_lattice_set_knobs: link " + std::to_string(i) +
                " does not name an existing multipole coefficient and a knob of the table");
      return XT_ERR_BAD_LATTICE;
    }
    const auto key = std::make_tuple(l.element, l.order, l.skew);
    if (!by_target.count(key)) order_seen.push_back(key);
    by_target[key].push_back(KnobLink{l.knob, 0, l.gain});
  }
  std::vector<KnobTarget> targets;
  std::vector<KnobLink> flat;
  for (const auto &key : order_seen) {
    const Elem &e = line.el[std::get<0>(key)];
    const int n = std::get<1>(key), skew = std::get<2>(key), big_n = static_cast<int>(e.aux);
    const double hxl = e.v[0], length = e.v[1];
    KnobTarget t{};
    // slots: (c[n], s[n]) pairs, n = N .. 0, from mult_slot0; wf sits in the record's second slot (xt_internal.h)
    t.off = lat->mult_slot0[std::get<0>(key)] + 16ull * static_cast<uint64_t>(big_n - n) + (skew ? 8ull : 0ull);
    t.wf_off = ~0ull;
    t.base = e.v[2 + (skew ? big_n + 1 : 0) + n];
    t.fact = 1.0;
    for (int k = 2; k <= n; ++k) t.fact *= static_cast<double>(k);
    t.hxl = 0.0;
    t.length = 1.0;
    if (n == 0 && !skew && hxl != 0.0) {
      t.hxl = hxl;
      if (length != 0.0) {
        t.wf_off = lat->mult_wf_off[std::get<0>(key)];
        t.length = length;
      }
    }
    t.first = static_cast<int32_t>(flat.size());
    t.count = static_cast<int32_t>(by_target[key].size());
    flat.insert(flat.end(), by_target[key].begin(), by_target[key].end());
    targets.push_back(t);
  }
  // build the new set first; the lattice keeps its previous knobs unless everything succeeded
  double *d_table = nullptr;
  void *d_targets = nullptr, *d_links = nullptr;
  auto fail = [&](cudaError_t e, const char *what) {
    cudaFree(d_table);
    cudaFree(d_targets);
    cudaFree(d_links);
    return cuda_fail(e, what);
  };
  cudaError_t e;
  const size_t tb = static_cast<size_t>(n_knobs) * n_steps * sizeof(double);
  if ((e = cudaMalloc(reinterpret_cast<void **>(&d_table), tb)) != cudaSuccess) return fail(e, "cudaMalloc(knob table)");
  if ((e = cudaMalloc(&d_targets, targets.size() * sizeof(KnobTarget))) != cudaSuccess)
    return fail(e, "cudaMalloc(knob targets)");
  if ((e = cudaMalloc(&d_links, flat.size() * sizeof(KnobLink))) != cudaSuccess)
    return fail(e, "cudaMalloc(knob links)");
  if ((e = cudaMemcpy(d_table, table, tb, cudaMemcpyHostToDevice)) != cudaSuccess)
    return fail(e, "cudaMemcpy(knob table)");
  if ((e = cudaMemcpy(d_targets, targets.data(), targets.size() * sizeof(KnobTarget), cudaMemcpyHostToDevice)) !=
      cudaSuccess)
    return fail(e, "cudaMemcpy(knob targets)");
  if ((e = cudaMemcpy(d_links, flat.data(), flat.size() * sizeof(KnobLink), cudaMemcpyHostToDevice)) != cudaSuccess)
    return fail(e, "cudaMemcpy(knob links)");
  drop_knobs(lat);
  lat->d_knob_table = d_table;
  lat->d_knob_targets = d_targets;
  lat->d_knob_links = d_links;
  lat->n_knob_targets = static_cast<int64_t>(targets.size());
  lat->n_knob_steps = n_steps;
  return XT_OK;
}

static int xt_track_knobs_impl(xt_lattice *lat, const xt_particles *p, int64_t n_part, int64_t n_turns,
                              int64_t step0, void *cuda_stream) {
  using namespace xt;
  if (!lat || !p || n_turns < 0) {
    set_error("xt_track_knobs: lat or p is NULL, or n_turns < 0");
    return XT_ERR_INVALID_ARG;
  }
  if (lat->n_knob_targets == 0) {
    set_error("xt_track_knobs: the lattice has no knobs (xt_lattice_set_knobs)");
    return XT_ERR_INVALID_ARG;
  }
  const int rc_dev = check_device(lat, "xt_track_knobs");  // before the first launch touches the image
  if (rc_dev != XT_OK) return rc_dev;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  xt_track_opts opts{};
  opts.compact_every = -1;
  int rc = XT_OK;
  for (int64_t j = 0; j < n_turns && rc == XT_OK; ++j) {
    const int64_t step = std::min<int64_t>(std::max<int64_t>(step0 + j, 0), lat->n_knob_steps - 1);
    rc = launch_apply(lat, step, 1, st);
    if (rc == XT_OK) rc = xt_track_ex(lat, p, n_part, 1, cuda_stream, &opts);
  }
  const int rc_restore = launch_apply(lat, 0, 0, st);  // the image goes back to its base values, whatever happened
  return rc != XT_OK ? rc : rc_restore;
}

// C ABI: no C++ exception may cross it (include/xt.h: "No exceptions, no abort()").  The bodies above use
// std::vector / std::map / std::string; a failed host allocation comes back as XT_ERR_NOMEM.
extern "C" int xt_lattice_set_knobs(xt_lattice *lat, const double *table, int32_t n_knobs, int64_t n_steps, const xt_knob_link *links, int64_t n_links) {
  return xt::guarded<int>([&] { return xt_lattice_set_knobs_impl(lat, table, n_knobs, n_steps, links, n_links); });
}

extern "C" int xt_track_knobs(xt_lattice *lat, const xt_particles *p, int64_t n_part, int64_t n_turns, int64_t step0, void *cuda_stream) {
  return xt::guarded<int>([&] { return xt_track_knobs_impl(lat, p, n_part, n_turns, step0, cuda_stream); });
}
