// Step C (loss compaction) and step H (survival histogram), SURVEY.md 8(a).
//
// Aperture elements "stop the tracking for the particles found to be outside"
// (PAPER.md:178).  A stopped particle is frozen, so it can be retired: every compact_every
// turns the alive particles are packed to the front of a working SoA (stable partition in ONE
// kernel: warp ballot + popc, block scan, single-pass look-back scan over the tiles) so that the
// tracking kernel's warps stay full; each retired particle is written straight to its final place
// in the caller's arrays through its origin index.  HBM-bound, 2 x n x 112 B per pass; measured
// 4.0-4.4 TB/s on 2e6 particles (profiles/r02_compaction_summary.md).
#include <atomic>
#include <string>

#include "xt_internal.h"

namespace xt {
namespace {

constexpr int kTile = 256;  // particles per CTA in the partition kernels

__device__ __forceinline__ void copy_particle(const xt_particles &dst, int64_t j, const xt_particles &src,
                                              int64_t i) {
  dst.x[j] = src.x[i];
  dst.px[j] = src.px[i];
  dst.y[j] = src.y[i];
  dst.py[j] = src.py[i];
  dst.zeta[j] = src.zeta[i];
  dst.delta[j] = src.delta[i];
  dst.ptau[j] = src.ptau[i];
  dst.rpp[j] = src.rpp[i];
  dst.rvv[j] = src.rvv[i];
  dst.s[j] = src.s[i];
  dst.at_turn[j] = src.at_turn[i];
  dst.state[j] = src.state[i];
  if (dst.at_element) dst.at_element[j] = src.at_element ? src.at_element[i] : 0;
}

// One pass, one kernel: stable partition with a single-pass ("decoupled look-back") scan over the tiles.
// Every CTA takes a ticket (tiles are then processed in ticket order whatever order the hardware starts
// CTAs in), counts its alive particles (ballot + popc), publishes the count, looks back over the tiles
// before it until it meets one whose inclusive prefix is known, publishes its own inclusive prefix and
// moves its particles: alive ones to dst[prefix + rank] (carrying their origin index), lost ones of a
// working set straight to their final place user[origin].  The last tile writes the new alive count.
// Status word of a tile: [epoch : 30][flag : 2][value : 32]; flag 1 = the tile's own count, 2 = inclusive
// prefix; the epoch (one per pass) makes words of earlier passes read as "not ready", so the array is
// cleared once per xt_track_ex call, not once per pass.  Reads 8 B (state) + 112 B per particle once,
// writes 112 B per particle once: the 2 x n x 112 B of SURVEY.md 8(a) row C plus the state read it
// repeats (the count must be known before the move).
constexpr uint64_t kFlagAggregate = 1, kFlagPrefix = 2;
__device__ __forceinline__ uint64_t pack_status(uint32_t epoch, uint64_t flag, uint32_t value) {
  return (static_cast<uint64_t>(epoch) << 34) | (flag << 32) | value;
}

__global__ void __launch_bounds__(kTile) partition_fused_kernel(xt_particles src, const int64_t *src_origin,
                                                                const int64_t *n_src_ptr, int64_t n_src_val,
                                                                xt_particles dst, int64_t *dst_origin,
                                                                xt_particles user, int retire_lost,
                                                                unsigned long long *status, unsigned int *ticket,
                                                                uint32_t epoch, int64_t *n_dst) {
  __shared__ int warp_counts[kTile / 32];
  __shared__ unsigned int s_tile;
  __shared__ uint32_t s_excl;
  if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
  __syncthreads();
  const unsigned int tile = s_tile;
  const int64_t n_src = n_src_ptr ? *n_src_ptr : n_src_val;
  const int64_t n_tiles_used = n_src > 0 ? (n_src + kTile - 1) / kTile : 1;  // tile 0 always reports
  if (static_cast<int64_t>(tile) >= n_tiles_used) {
    if (tile == gridDim.x - 1 && threadIdx.x == 0) *ticket = 0;  // the last ticket holder resets the counter
    return;
  }
  const int64_t i = static_cast<int64_t>(tile) * kTile + threadIdx.x;
  const bool in_range = i < n_src;
  // the whole record goes into registers before the scan: the loads are in flight while the tile waits for
  // its prefix
  double f[10] = {};
  int64_t at_turn = 0, state = 0, at_element = 0, origin = 0;
  if (in_range) {
    state = src.state[i];
    f[0] = src.x[i];
    f[1] = src.px[i];
    f[2] = src.y[i];
    f[3] = src.py[i];
    f[4] = src.zeta[i];
    f[5] = src.delta[i];
    f[6] = src.ptau[i];
    f[7] = src.rpp[i];
    f[8] = src.rvv[i];
    f[9] = src.s[i];
    at_turn = src.at_turn[i];
    at_element = src.at_element ? src.at_element[i] : 0;
    origin = src_origin ? src_origin[i] : i;
  }
  const bool alive = in_range && (state == 1);
  const unsigned ballot = __ballot_sync(0xffffffffu, alive);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) warp_counts[warp] = __popc(ballot);
  __syncthreads();
  int before = 0, total = 0;
#pragma unroll
  for (int w = 0; w < kTile / 32; ++w) {
    const int c = warp_counts[w];
    if (w < warp) before += c;
    total += c;
  }
  if (warp == 0) {
    // publish the tile's own count, then look back (32 predecessors at a time)
    uint32_t excl = 0;
    if (tile == 0) {
      if (lane == 0) atomicExch(&status[0], pack_status(epoch, kFlagPrefix, static_cast<uint32_t>(total)));
    } else {
      if (lane == 0) atomicExch(&status[tile], pack_status(epoch, kFlagAggregate, static_cast<uint32_t>(total)));
      int64_t look = static_cast<int64_t>(tile) - 1;
      bool done = false;
      while (!done) {
        const int64_t k = look - lane;
        uint64_t w = 0;
        uint64_t flag = kFlagPrefix;  // lanes before tile 0 read as a zero prefix
        if (k >= 0) {
          do {
            w = atomicAdd(&status[k], 0ull);  // volatile read through L2
            flag = ((w >> 34) == epoch) ? ((w >> 32) & 3u) : 0u;
          } while (flag == 0);
        }
        const unsigned has_prefix = __ballot_sync(0xffffffffu, flag == kFlagPrefix);
        const int first = __ffs(has_prefix) - 1;  // nearest tile with a known inclusive prefix (there is one if k < 0 anywhere)
        const uint32_t v = (k >= 0 && (first < 0 || lane <= first)) ? static_cast<uint32_t>(w) : 0u;
        excl += __reduce_add_sync(0xffffffffu, v);
        if (first >= 0) done = true;
        else look -= 32;
      }
      if (lane == 0) atomicExch(&status[tile], pack_status(epoch, kFlagPrefix, excl + static_cast<uint32_t>(total)));
    }
    if (lane == 0) {
      s_excl = excl;
      if (static_cast<int64_t>(tile) == n_tiles_used - 1) *n_dst = static_cast<int64_t>(excl) + total;
      if (tile == gridDim.x - 1) *ticket = 0;
    }
  }
  __syncthreads();
  const int rank = before + __popc(ballot & ((1u << lane) - 1u));
  if (!in_range || (!alive && !retire_lost)) return;
  const xt_particles &o = alive ? dst : user;
  const int64_t j = alive ? static_cast<int64_t>(s_excl) + rank : origin;
  o.x[j] = f[0];
  o.px[j] = f[1];
  o.y[j] = f[2];
  o.py[j] = f[3];
  o.zeta[j] = f[4];
  o.delta[j] = f[5];
  o.ptau[j] = f[6];
  o.rpp[j] = f[7];
  o.rvv[j] = f[8];
  o.s[j] = f[9];
  o.at_turn[j] = at_turn;
  o.state[j] = state;
  if (o.at_element) o.at_element[j] = at_element;
  if (alive) dst_origin[j] = origin;
}

__global__ void __launch_bounds__(kTile) scatter_back_kernel(xt_particles src, const int64_t *src_origin,
                                                             const int64_t *n_src_ptr, xt_particles user) {
  const int64_t n_src = *n_src_ptr;
  const int64_t i = static_cast<int64_t>(blockIdx.x) * kTile + threadIdx.x;
  if (i >= n_src) return;
  copy_particle(user, src_origin[i], src, i);
}

// Step H.  Shared-memory histogram per CTA, one global atomic per non-empty bin per CTA.
__global__ void __launch_bounds__(256) histogram_kernel(const int64_t *__restrict__ at_turn,
                                                        const int64_t *__restrict__ state, int64_t n,
                                                        int64_t bin_width, int n_bins,
                                                        unsigned long long *hist) {
  extern __shared__ unsigned int sh[];
  for (int b = threadIdx.x; b <= n_bins; b += blockDim.x) sh[b] = 0u;
  __syncthreads();
  const int64_t stride = static_cast<int64_t>(gridDim.x) * blockDim.x;
  for (int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; i < n; i += stride) {
    int b;
    if (state[i] == 1) {
      b = n_bins;
    } else {
      int64_t q = at_turn[i] / bin_width;
      if (q < 0) q = 0;
      if (q > n_bins - 1) q = n_bins - 1;
      b = static_cast<int>(q);
    }
    // neighbouring particles of an amplitude scan mostly share a bin: one shared-memory atomic per
    // distinct bin of the warp instead of one per particle
    const unsigned active = __activemask();
    const unsigned same = __match_any_sync(active, b);
    if ((__ffs(same) - 1) == static_cast<int>(threadIdx.x & 31)) atomicAdd(&sh[b], static_cast<unsigned int>(__popc(same)));
  }
  __syncthreads();
  for (int b = threadIdx.x; b <= n_bins; b += blockDim.x)
    if (sh[b]) atomicAdd(&hist[b], static_cast<unsigned long long>(sh[b]));
}

size_t align256(size_t v) { return (v + 255) & ~static_cast<size_t>(255); }

}  // namespace

size_t compaction_workspace_bytes(int64_t n_part) {
  const size_t arr = align256(static_cast<size_t>(n_part) * 8);
  const int64_t n_tiles = (n_part + kTile - 1) / kTile;
  return 2 * 14 * arr + align256(static_cast<size_t>(n_tiles) * 8) + 256;
}

void plan_compaction(void *ws, int64_t n_part, CompactPlan &plan) {
  unsigned char *at = static_cast<unsigned char *>(ws);
  const size_t arr = align256(static_cast<size_t>(n_part) * 8);
  auto take = [&]() {
    void *r = at;
    at += arr;
    return r;
  };
  for (int k = 0; k < 2; ++k) {
    xt_particles &p = plan.w[k].p;
    p.x = static_cast<double *>(take());
    p.px = static_cast<double *>(take());
    p.y = static_cast<double *>(take());
    p.py = static_cast<double *>(take());
    p.zeta = static_cast<double *>(take());
    p.delta = static_cast<double *>(take());
    p.ptau = static_cast<double *>(take());
    p.rpp = static_cast<double *>(take());
    p.rvv = static_cast<double *>(take());
    p.s = static_cast<double *>(take());
    p.at_turn = static_cast<int64_t *>(take());
    p.state = static_cast<int64_t *>(take());
    p.at_element = static_cast<int64_t *>(take());
    p.particle_id = nullptr;
    plan.w[k].origin = static_cast<int64_t *>(take());
  }
  plan.n_tiles = (n_part + kTile - 1) / kTile;
  plan.status = reinterpret_cast<unsigned long long *>(at);
  at += align256(static_cast<size_t>(plan.n_tiles) * 8);
  plan.counter[0] = reinterpret_cast<int64_t *>(at);
  plan.counter[1] = plan.counter[0] + 1;
  plan.ticket = reinterpret_cast<unsigned int *>(plan.counter[0] + 2);
  plan.n_active = plan.counter[0];
  plan.epoch = 0;
}

int launch_partition(CompactPlan &plan, const xt_particles &src, const int64_t *src_origin, bool src_is_user,
                     int64_t n_part, const WorkSet &dst, const xt_particles &user, cudaStream_t st) {
  if (n_part <= 0) return XT_OK;
  if (plan.epoch == 0) {  // first pass of the call: the status words and the ticket start from zero
    XT_CUDA(cudaMemsetAsync(plan.status, 0, static_cast<size_t>(plan.n_tiles) * 8, st));
    XT_CUDA(cudaMemsetAsync(plan.counter[0], 0, 32, st));
  }
  plan.epoch += 1;
  // the pass reads the extent of src from one counter and writes the new alive count to the other
  int64_t *n_in = plan.n_active;
  int64_t *n_out = (n_in == plan.counter[0]) ? plan.counter[1] : plan.counter[0];
  partition_fused_kernel<<<static_cast<unsigned>(plan.n_tiles), kTile, 0, st>>>(
      src, src_origin, src_is_user ? nullptr : n_in, n_part, dst.p, dst.origin, user, src_is_user ? 0 : 1,
      plan.status, plan.ticket, plan.epoch, n_out);
  XT_CUDA(cudaGetLastError());
  plan.n_active = n_out;
  count_launch();
  return XT_OK;
}

int launch_scatter_back(const CompactPlan &plan, const WorkSet &src, int64_t n_part, const xt_particles &user,
                        cudaStream_t st) {
  if (n_part <= 0) return XT_OK;
  scatter_back_kernel<<<static_cast<unsigned>(plan.n_tiles), kTile, 0, st>>>(src.p, src.origin, plan.n_active,
                                                                            user);
  XT_CUDA(cudaGetLastError());
  count_launch();
  return XT_OK;
}

int launch_histogram(const int64_t *at_turn, const int64_t *state, int64_t n, int64_t bin_width, int64_t n_bins,
                     int64_t *hist, cudaStream_t st) {
  XT_CUDA(cudaMemsetAsync(hist, 0, static_cast<size_t>(n_bins + 1) * 8, st));
  if (n <= 0) return XT_OK;
  int64_t grid = (n + 255) / 256;
  if (grid > 148 * 2) grid = 148 * 2;  // few CTAs: the global atomics at the end all hit the same n_bins + 1 words
  histogram_kernel<<<static_cast<unsigned>(grid), 256, static_cast<size_t>(n_bins + 1) * 4, st>>>(
      at_turn, state, n, bin_width, static_cast<int>(n_bins), reinterpret_cast<unsigned long long *>(hist));
  XT_CUDA(cudaGetLastError());
  count_launch();
  return XT_OK;
}

}  // namespace xt

// ------------------------------------------------------------------ xt_track_static (include/xt.h)
// Tracking with loss compaction for callers that may not allocate (CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc): the whole scratch of step C -- two working sets of 14 arrays, the tile
// status words of the single-pass scan, the ticket and the two counters -- lives in ONE file-scope device
// array of fixed size instead of a cudaMallocAsync block.  Every GPU that loads the library holds the
// array (7.0 MiB) until the process exits.  All calls share it: it keeps the previous call's bytes, two
// calls that overlap on the GPU race (see the header).  What must start at zero (status words, ticket,
// counters) is cleared by the first pass of every call (launch_partition, plan.epoch == 0); the working
// sets are written by a pass before anything reads them.
namespace xt {
namespace {

constexpr int64_t kStaticMaxParticles = XT_TRACK_STATIC_MAX_PARTICLES;
constexpr size_t up256(size_t v) { return (v + 255) & ~static_cast<size_t>(255); }
constexpr size_t kStaticBytes = 2 * 14 * up256(static_cast<size_t>(kStaticMaxParticles) * 8) +
                                up256(static_cast<size_t>((kStaticMaxParticles + kTile - 1) / kTile) * 8) + 256;
static_assert(kStaticBytes <= (8u << 20), "the static workspace is meant to stay modest");

static __device__ __align__(256) unsigned char g_static_workspace[kStaticBytes];

// In host code `g_static_workspace` is only a handle of the symbol, not a device address: the address
// comes from cudaGetSymbolAddress, once per device, with that device current.
constexpr int kMaxDevices = 64;
std::atomic<void *> g_static_address[kMaxDevices];

int static_workspace_address(void **out) {
  int dev = -1;
  XT_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) {
    set_error("xt_track_static: device ordinal out of range");
    return XT_ERR_INVALID_ARG;
  }
  void *ptr = g_static_address[dev].load(std::memory_order_acquire);
  if (!ptr) {
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_workspace);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(static workspace)");
    if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255u)) {
      set_error("xt_track_static: the static workspace has no 256-byte aligned device address");
      return XT_ERR_CUDA;
    }
    g_static_address[dev].store(ptr, std::memory_order_release);
  }
  *out = ptr;
  return XT_OK;
}

}  // namespace
}  // namespace xt

extern "C" int xt_track_static(const xt_lattice *lat, const xt_particles *p, int64_t n_part, int64_t n_turns,
                               void *cuda_stream, const xt_track_opts *opts) {
  return xt::guarded<int>([&] {
    if (!lat || !p) {
      xt::set_error("xt_track_static: NULL lattice or particles");
      return static_cast<int>(XT_ERR_INVALID_ARG);
    }
    if (n_part > xt::kStaticMaxParticles) {
      xt::set_error("xt_track_static: n_part = " + std::to_string(n_part) + " exceeds XT_TRACK_STATIC_MAX_PARTICLES = " +
                    std::to_string(xt::kStaticMaxParticles) +
                    ", all the static device workspace holds; use xt_track_ex with xt_track_opts.workspace");
      return static_cast<int>(XT_ERR_INVALID_ARG);
    }
    if (opts && (opts->workspace || opts->workspace_bytes || opts->stats)) {
      xt::set_error("xt_track_static: xt_track_opts.workspace / .stats must be NULL (the workspace is the library's "
                    "static array; the stats record allocates)");
      return static_cast<int>(XT_ERR_INVALID_ARG);
    }
    int rc = xt::check_device(lat, "xt_track_static");
    if (rc != XT_OK) return rc;
    if (xt::compaction_workspace_bytes(xt::kStaticMaxParticles) > xt::kStaticBytes) {
      xt::set_error("xt_track_static: internal error, the static workspace is smaller than step C needs");
      return static_cast<int>(XT_ERR_CUDA);
    }
    void *ws = nullptr;
    if ((rc = xt::static_workspace_address(&ws)) != XT_OK) return rc;
    xt_track_opts o = opts ? *opts : xt_track_opts{};
    o.workspace = ws;  // a device address; the partition and tracking kernels receive pointers cut from it
    o.workspace_bytes = xt::kStaticBytes;
    return xt_track_ex(lat, p, n_part, n_turns, cuda_stream, &o);
  });
}
