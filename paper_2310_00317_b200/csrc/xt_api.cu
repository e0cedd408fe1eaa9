// C-ABI entry points that orchestrate the kernels (include/xt.h): xt_track / xt_track_ex
// (launch chunking + periodic compaction), xt_track_host (end-to-end with host buffers),
// the init helper, the survival histogram, the FMA microbenchmark and error reporting.
#include <atomic>
#include <string>
#include <vector>

#include "xt_internal.h"

namespace xt {
namespace {
thread_local std::string g_error;
std::atomic<int64_t> g_launches{0};
}  // namespace

void set_error(const std::string &msg) { g_error = msg; }

int cuda_fail(cudaError_t e, const char *what) {
  g_error = std::string(what) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")";
  return e == cudaErrorMemoryAllocation ? XT_ERR_NOMEM : XT_ERR_CUDA;
}

void count_launch(int64_t n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

int check_device(const xt_lattice *lat, const char *fn) {
  int dev = -1;
  XT_CUDA(cudaGetDevice(&dev));
  if (!lat || dev != lat->device) {  // the lattice image lives on the device it was created on
    set_error(std::string(fn) + ": the current CUDA device is not the one the lattice was created on");
    return XT_ERR_INVALID_ARG;
  }
  return XT_OK;
}

namespace {

int check_particles(const char *fn, const xt_lattice *lat, const xt_particles *p, int64_t n_part) {
  if (!lat || !p || n_part < 0) {
    set_error(std::string(fn) + ": NULL lattice/particles or negative n_part");
    return XT_ERR_INVALID_ARG;
  }
  if (n_part > 0 && (!p->x || !p->px || !p->y || !p->py || !p->zeta || !p->delta || !p->ptau || !p->rpp ||
                     !p->rvv || !p->s || !p->at_turn || !p->state)) {
    set_error(std::string(fn) + ": a required particle array is NULL (only particle_id, at_element may be)");
    return XT_ERR_INVALID_ARG;
  }
  return check_device(lat, fn);
}

// Launch shape of the tracking kernel: threads per CTA, particles per thread, and where the cold
// per-particle state lives.  Auto rule (measured on B200, profiles/r02_shape_sweep.md): 128-thread CTAs.
// The static shape for many waves of particles: 4 per thread, cold state in shared memory, 4 CTAs per
// SM at <= 128 registers, every CTA owning its share for the whole launch.  Up to ~12 000 per SM, when the
// launch is long enough for the balanced mode (xt_track.cu: one CTA per (group, block of turns) item, a
// queue of ready groups): the cold state in registers, 2 per thread up to 1024 per SM, 3 above; full
// warps and an SM that is never short of a CTA beat the static shapes by 16-30 % there (configs[2]: 0.522 ->
// 0.610 of the DFMA peak; 150 000 particles on the configs[3] lattice: 0.477 -> 0.619; 10^6: 0.608 ->
// 0.644; 2 * 10^6: equal).  Beyond that, on thin lattices: 4 per thread in registers at a 168-register cap,
// still balanced (configs[3]: 0.659 -> 0.662).  Launches too short for that: 2 per thread / registers up to 768 per SM
// (configs[2] statically: 0.524 against 0.511 for 3 per thread), 3 per thread / shared memory up to 4096,
// 4 above.  Below ~100 particles per SM one per thread keeps more warps alive.
struct Shape {
  int block, ppt;
  bool cold_in_regs;
};
int resolve_shape(const xt_track_opts *o, const xt_lattice *lat, int64_t n_part, bool can_balance, bool compacting,
                  Shape *sh) {
  const int64_t per_sm = n_part / (lat->n_sm > 0 ? lat->n_sm : 1);
  // with compaction n_part is only the bound of what is still alive: lean towards the balanced shapes
  const int64_t balanced_up_to = compacting ? 16384 : 12288;
  int auto_ppt = 4, auto_block = 128;
  bool auto_regs = false;
  if (per_sm < 4096) auto_ppt = 3;
  if (can_balance && per_sm > balanced_up_to && !lat->extended) auto_regs = true;  // 4 per thread, balanced
  if (can_balance && per_sm <= balanced_up_to) {
    auto_ppt = 3;  // (4 per thread / registers: +2 % on the configs[3] lattice, -0.7 % on configs[4]; by option)
    auto_regs = true;
  }
  if (per_sm <= 768 || (can_balance && per_sm <= 1024)) {
    auto_ppt = 2;
    auto_regs = true;
  }
  if (per_sm < 96) {
    auto_ppt = 1;
    auto_block = 32;
    auto_regs = false;
  }
  sh->ppt = (o && o->particles_per_thread) ? o->particles_per_thread : auto_ppt;
  sh->block = (o && o->block_size) ? o->block_size : auto_block;
  const int want_regs = o ? o->cold_in_registers : 0;
  if (want_regs > 0)
    sh->cold_in_regs = true;
  else if (want_regs < 0)
    sh->cold_in_regs = false;
  else
    sh->cold_in_regs = auto_regs;
  if (sh->ppt < 1 || sh->ppt > 4) {
    set_error("xt_track_ex: particles_per_thread must be 0 (auto), 1, 2, 3 or 4");
    return XT_ERR_INVALID_ARG;
  }
  if (sh->block < 32 || sh->block > 256 || (sh->block % 32) != 0) {
    set_error("xt_track_ex: block_size must be a multiple of 32 in [32, 256]");
    return XT_ERR_INVALID_ARG;
  }
  return XT_OK;
}

// Optional timing of one xt_track_ex call (xt_track_stats): events around every tracking launch and every
// compaction pass; the alive count behind each pass is logged by an 8-byte device copy.  All host work
// happens in finish(), after one stream synchronisation.  Inactive (stats == nullptr) it does nothing.
class StatsTimer {
 public:
  StatsTimer(xt_track_stats *stats, cudaStream_t st) : stats_(stats), st_(st) {}
  ~StatsTimer() {
    for (auto &e : ev_) {
      cudaEventDestroy(e.a);
      cudaEventDestroy(e.b);
    }
    if (d_log_) cudaFree(d_log_);
  }
  void begin() {
    if (!stats_) return;
    Span s{};
    s.kind = -1;  // until its end is recorded
    if (cudaEventCreate(&s.a) != cudaSuccess) {
      failed_ = true;
      return;
    }
    if (cudaEventCreate(&s.b) != cudaSuccess) {
      cudaEventDestroy(s.a);
      failed_ = true;
      return;
    }
    cudaEventRecord(s.a, st_);
    ev_.push_back(s);
  }
  void end_track() { end(0, nullptr); }
  void end_pass(const int64_t *d_n_active) { end(1, d_n_active); }
  void end_scatter() { end(2, nullptr); }
  int finish(int64_t n_part) {
    if (!stats_) return XT_OK;
    XT_CUDA(cudaStreamSynchronize(st_));
    if (failed_) {  // an event could not be created: the tracking itself is complete, the record is not
      set_error("xt_track_ex: could not create the CUDA events of xt_track_stats");
      return XT_ERR_CUDA;
    }
    xt_track_stats &o = *stats_;
    o = xt_track_stats{};
    std::vector<int64_t> log(n_pass_);
    if (n_pass_) XT_CUDA(cudaMemcpy(log.data(), d_log_, sizeof(int64_t) * n_pass_, cudaMemcpyDeviceToHost));
    int64_t n_in = n_part, pass = 0;
    for (const Span &s : ev_) {
      float ms = 0.f;
      XT_CUDA(cudaEventElapsedTime(&ms, s.a, s.b));
      if (s.kind == 0) {
        o.n_track_launches++;
        o.track_ms += ms;
      } else if (s.kind == 1) {
        const int64_t n_out = log[pass];
        if (pass < XT_STATS_MAX_PASSES) {
          o.pass_n_in[pass] = n_in;
          o.pass_n_out[pass] = n_out;
          o.pass_ms[pass] = ms;
        }
        o.compact_ms += ms;
        o.compact_bytes += 2.0 * 112.0 * static_cast<double>(n_in);
        n_in = n_out;
        ++pass;
      } else {
        o.scatter_ms += ms;
        o.scatter_bytes += 2.0 * 112.0 * static_cast<double>(n_in);
      }
    }
    o.n_passes = pass;
    return XT_OK;
  }

 private:
  struct Span {
    cudaEvent_t a, b;
    int kind;
  };
  void end(int kind, const int64_t *d_n_active) {
    if (!stats_ || failed_ || ev_.empty() || ev_.back().kind != -1) return;
    ev_.back().kind = kind;
    cudaEventRecord(ev_.back().b, st_);
    if (kind == 1 && d_n_active) {
      if (!d_log_) cudaMalloc(reinterpret_cast<void **>(&d_log_), sizeof(int64_t) * kMaxLog);
      if (d_log_ && n_pass_ < kMaxLog)
        cudaMemcpyAsync(d_log_ + n_pass_++, d_n_active, sizeof(int64_t), cudaMemcpyDeviceToDevice, st_);
    }
  }
  static constexpr int kMaxLog = 1 << 16;
  xt_track_stats *stats_;
  cudaStream_t st_;
  std::vector<Span> ev_;
  int64_t *d_log_ = nullptr;
  int n_pass_ = 0;
  bool failed_ = false;
};

}  // namespace
}  // namespace xt

static int xt_track_ex_impl(const xt_lattice *lat, const xt_particles *p, int64_t n_part, int64_t n_turns,
                           void *cuda_stream, const xt_track_opts *opts) {
  int rc = xt::check_particles("xt_track", lat, p, n_part);
  if (rc != XT_OK) return rc;
  if (n_turns < 0) {
    xt::set_error("xt_track: negative n_turns");
    return XT_ERR_INVALID_ARG;
  }
  if (opts && opts->turns_per_launch < 0) {
    xt::set_error("xt_track_ex: negative turns_per_launch");
    return XT_ERR_INVALID_ARG;
  }
  if (n_part == 0 || n_turns == 0) return XT_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

  // compaction period (step C): only lattices with apertures can lose particles
  int64_t period = 0;
  const int64_t want = opts ? opts->compact_every : 0;
  if (lat->info.has_aperture && want >= 0) {
    const int64_t pr = want > 0 ? want : 1000;
    if (n_turns > pr) period = pr;
  }
  const int64_t tpl_opt = opts ? opts->turns_per_launch : 0;
  // the balanced mode needs launches of several blocks of turns and a particle count known to the host
  const int64_t launch_turns = (tpl_opt > 0 && tpl_opt < n_turns) ? tpl_opt : n_turns;
  const int64_t kernel_turns = (period > 0 && launch_turns > period) ? period : launch_turns;
  const bool can_balance = xt::balance_pays(lat, kernel_turns, opts ? opts->balance : 0);
  xt::Shape sh{};
  if ((rc = xt::resolve_shape(opts, lat, n_part, can_balance, period > 0, &sh)) != XT_OK) return rc;

  xt::StatsTimer tm(opts ? opts->stats : nullptr, st);
  if (period == 0) {
    // Balanced mode of the shapes with the cold state in registers (xt_track.cu): needs two counters and one
    // word per item, from the caller's workspace if there is one, else stream-ordered.
    const int balance = opts ? opts->balance : 0;
    unsigned int *queue = nullptr;
    bool own_queue = false;
    if (sh.cold_in_regs && can_balance) {
      const size_t qb = xt::balance_scratch_bytes(n_part, sh.block, sh.ppt);
      if (opts && opts->workspace) {
        if (opts->workspace_bytes >= qb && !(reinterpret_cast<uintptr_t>(opts->workspace) & 255u)) {
          queue = static_cast<unsigned int *>(opts->workspace);
        } else if (balance > 0) {
          xt::set_error("xt_track_ex: workspace too small for the balanced mode (xt_track_workspace_bytes is enough) or not 256-byte aligned");
          return XT_ERR_INVALID_ARG;
        }
      } else {
        XT_CUDA(cudaMallocAsync(reinterpret_cast<void **>(&queue), qb, st));
        own_queue = true;
      }
    } else if (balance > 0) {
      xt::set_error("xt_track_ex: balance > 0 needs the cold state in registers (cold_in_registers = 1, or the auto shape of small ensembles)");
      return XT_ERR_INVALID_ARG;
    }
    auto done = [&](int code) {
      if (own_queue) cudaFreeAsync(queue, st);
      return code;
    };
    const int64_t tpl = tpl_opt > 0 ? tpl_opt : n_turns;
    for (int64_t done_turns = 0; done_turns < n_turns;) {
      const int64_t k = (n_turns - done_turns < tpl) ? n_turns - done_turns : tpl;
      tm.begin();
      if ((rc = xt::launch_track(lat, *p, n_part, nullptr, k, sh.block, sh.ppt, sh.cold_in_regs, st, queue, balance)) != XT_OK)
        return done(rc);
      tm.end_track();
      done_turns += k;
    }
    return done(tm.finish(n_part));
  }

  void *ws = opts ? opts->workspace : nullptr;
  const size_t c_bytes = xt::compaction_workspace_bytes(n_part);
  // the balanced mode's queue sits behind the working sets when the shape can use it and there is room
  const int balance = opts ? opts->balance : 0;
  size_t q_bytes = (sh.cold_in_regs && can_balance) ? xt::balance_scratch_bytes(n_part, sh.block, sh.ppt) : 0;
  const bool own_ws = (ws == nullptr);
  if (!own_ws && (opts->workspace_bytes < c_bytes || (reinterpret_cast<uintptr_t>(ws) & 255u))) {
    xt::set_error("xt_track_ex: workspace too small (see xt_track_workspace_bytes) or not 256-byte aligned");
    return XT_ERR_INVALID_ARG;
  }
  if (!own_ws && opts->workspace_bytes < c_bytes + q_bytes) {
    if (balance > 0) {
      xt::set_error("xt_track_ex: workspace too small for the balanced mode with this launch shape");
      return XT_ERR_INVALID_ARG;
    }
    q_bytes = 0;
  }
  if (balance > 0 && !sh.cold_in_regs) {
    xt::set_error("xt_track_ex: balance > 0 needs the cold state in registers (cold_in_registers = 1, or the auto shape of small ensembles)");
    return XT_ERR_INVALID_ARG;
  }
  if (own_ws) XT_CUDA(cudaMallocAsync(&ws, c_bytes + q_bytes, st));
  unsigned int *queue = q_bytes ? reinterpret_cast<unsigned int *>(static_cast<unsigned char *>(ws) + c_bytes) : nullptr;
  xt::CompactPlan plan;
  xt::plan_compaction(ws, n_part, plan);
  auto bail = [&](int code) {
    if (own_ws) cudaFreeAsync(ws, st);
    return code;
  };
  // initial partition: alive particles of the caller's arrays -> working set 0
  tm.begin();
  if ((rc = xt::launch_partition(plan, *p, nullptr, true, n_part, plan.w[0], *p, st)) != XT_OK) return bail(rc);
  tm.end_pass(plan.n_active);
  int cur = 0;
  const int64_t tpl = (tpl_opt > 0 && tpl_opt < period) ? tpl_opt : period;
  int64_t since = 0;
  for (int64_t done = 0; done < n_turns;) {
    int64_t k = n_turns - done;
    if (k > tpl) k = tpl;
    if (k > period - since) k = period - since;
    tm.begin();
    if ((rc = xt::launch_track(lat, plan.w[cur].p, n_part, plan.n_active, k, sh.block, sh.ppt, sh.cold_in_regs, st, queue,
                               balance)) != XT_OK)
      return bail(rc);
    tm.end_track();
    done += k;
    since += k;
    if (since == period && done < n_turns) {
      tm.begin();
      if ((rc = xt::launch_partition(plan, plan.w[cur].p, plan.w[cur].origin, false, n_part, plan.w[1 - cur], *p,
                                     st)) != XT_OK)
        return bail(rc);
      tm.end_pass(plan.n_active);
      cur = 1 - cur;
      since = 0;
    }
  }
  tm.begin();
  if ((rc = xt::launch_scatter_back(plan, plan.w[cur], n_part, *p, st)) != XT_OK) return bail(rc);
  tm.end_scatter();
  if ((rc = tm.finish(n_part)) != XT_OK) return bail(rc);
  if (own_ws) XT_CUDA(cudaFreeAsync(ws, st));
  return XT_OK;
}

extern "C" uint64_t xt_track_workspace_bytes(int64_t n_part) {
  // the working sets of step C, and behind them the queue of the balanced mode for the auto shapes
  return n_part > 0 ? static_cast<uint64_t>(xt::compaction_workspace_bytes(n_part) + xt::balance_scratch_bytes(n_part, 128, 2))
                    : 0;
}

extern "C" int xt_track(const xt_lattice *lat, const xt_particles *p, int64_t n_part, int64_t n_turns,
                        void *cuda_stream) {
  return xt_track_ex(lat, p, n_part, n_turns, cuda_stream, nullptr);
}

static int xt_track_host_impl(const xt_lattice *lat, const xt_particles *hp, int64_t n_part, int64_t n_turns,
                             void *cuda_stream, const xt_track_opts *opts) {
  int rc = xt::check_particles("xt_track_host", lat, hp, n_part);
  if (rc != XT_OK) return rc;
  if (n_turns < 0) {
    xt::set_error("xt_track_host: negative n_turns");
    return XT_ERR_INVALID_ARG;
  }
  if (n_part == 0 || n_turns == 0) return XT_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const size_t arr = (static_cast<size_t>(n_part) * 8 + 255) & ~static_cast<size_t>(255);
  const int n_arr = 13;
  unsigned char *buf = nullptr;
  XT_CUDA(cudaMallocAsync(reinterpret_cast<void **>(&buf), arr * n_arr, st));
  void *host[13] = {hp->x,   hp->px,  hp->y, hp->py,      hp->zeta,  hp->delta,     hp->ptau,
                    hp->rpp, hp->rvv, hp->s, hp->at_turn, hp->state, hp->at_element};
  void *dev[13];
  for (int k = 0; k < n_arr; ++k) dev[k] = buf + arr * k;
  auto bail = [&](int code) {
    cudaFreeAsync(buf, st);
    return code;
  };
  for (int k = 0; k < n_arr; ++k) {
    if (!host[k]) continue;  // at_element is optional
    cudaError_t e = cudaMemcpyAsync(dev[k], host[k], static_cast<size_t>(n_part) * 8, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return bail(xt::cuda_fail(e, "cudaMemcpyAsync(H2D)"));
  }
  xt_particles dp{};
  dp.x = static_cast<double *>(dev[0]);
  dp.px = static_cast<double *>(dev[1]);
  dp.y = static_cast<double *>(dev[2]);
  dp.py = static_cast<double *>(dev[3]);
  dp.zeta = static_cast<double *>(dev[4]);
  dp.delta = static_cast<double *>(dev[5]);
  dp.ptau = static_cast<double *>(dev[6]);
  dp.rpp = static_cast<double *>(dev[7]);
  dp.rvv = static_cast<double *>(dev[8]);
  dp.s = static_cast<double *>(dev[9]);
  dp.at_turn = static_cast<int64_t *>(dev[10]);
  dp.state = static_cast<int64_t *>(dev[11]);
  dp.at_element = hp->at_element ? static_cast<int64_t *>(dev[12]) : nullptr;
  dp.particle_id = nullptr;
  if ((rc = xt_track_ex(lat, &dp, n_part, n_turns, cuda_stream, opts)) != XT_OK) return bail(rc);
  for (int k = 0; k < n_arr; ++k) {
    if (!host[k]) continue;
    cudaError_t e = cudaMemcpyAsync(host[k], dev[k], static_cast<size_t>(n_part) * 8, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return bail(xt::cuda_fail(e, "cudaMemcpyAsync(D2H)"));
  }
  XT_CUDA(cudaFreeAsync(buf, st));
  XT_CUDA(cudaStreamSynchronize(st));
  return XT_OK;
}

extern "C" int xt_particles_init_derived(const xt_lattice *lat, const xt_particles *p, int64_t n_part,
                                         void *cuda_stream) {
  if (!lat || !p || n_part < 0 || (n_part > 0 && (!p->delta || !p->ptau || !p->rpp || !p->rvv))) {
    xt::set_error("xt_particles_init_derived: NULL argument or negative n_part");
    return XT_ERR_INVALID_ARG;
  }
  return xt::launch_init_derived(lat, *p, n_part, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int xt_survival_histogram(const int64_t *at_turn, const int64_t *state, int64_t n_part,
                                     int64_t bin_width, int64_t n_bins, int64_t *hist, void *cuda_stream) {
  if (!hist || n_part < 0 || bin_width <= 0 || n_bins <= 0 || n_bins > 8192 ||
      (n_part > 0 && (!at_turn || !state))) {
    xt::set_error("xt_survival_histogram: invalid argument (need bin_width > 0, 0 < n_bins <= 8192)");
    return XT_ERR_INVALID_ARG;
  }
  return xt::launch_histogram(at_turn, state, n_part, bin_width, n_bins, hist,
                              static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int xt_fp64_fma_peak(double *flops_per_s, double *ms, void *cuda_stream) {
  return xt::run_fma_peak(flops_per_s, ms, 0, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int xt_fp64_fma_peak_sweep_size(void) { return xt::fma_peak_sweep_size(); }

extern "C" int xt_fp64_fma_peak_sweep(int index, double *flops_per_s, double *ms, int *desc, void *cuda_stream) {
  return xt::run_fma_peak_shape(index, flops_per_s, ms, desc, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int xt_fp64_fma_probe(int pattern, double *flops_per_s, double *ms, void *cuda_stream) {
  return xt::run_fma_peak(flops_per_s, ms, pattern, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int64_t xt_launch_count(void) { return xt::g_launches.load(std::memory_order_relaxed); }

extern "C" const char *xt_last_error(void) { return xt::g_error.c_str(); }

extern "C" const char *xt_build_info(void) {
#ifdef XT_FMAD_OFF
  return "libxt_b200 sm_100a fmad=false (validation build)";
#else
  return "libxt_b200 sm_100a fmad=true";
#endif
}

// C ABI: no C++ exception may cross it (include/xt.h: "No exceptions, no abort()").  The bodies above use
// std::vector / std::map / std::string; a failed host allocation comes back as XT_ERR_NOMEM.
extern "C" int xt_track_ex(const xt_lattice *lat, const xt_particles *p, int64_t n_part, int64_t n_turns, void *cuda_stream, const xt_track_opts *opts) {
  return xt::guarded<int>([&] { return xt_track_ex_impl(lat, p, n_part, n_turns, cuda_stream, opts); });
}

extern "C" int xt_track_host(const xt_lattice *lat, const xt_particles *hp, int64_t n_part, int64_t n_turns, void *cuda_stream, const xt_track_opts *opts) {
  return xt::guarded<int>([&] { return xt_track_host_impl(lat, hp, n_part, n_turns, cuda_stream, opts); });
}
