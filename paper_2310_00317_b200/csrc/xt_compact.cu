// Step C (loss compaction) and step H (survival histogram), SURVEY.md 8(a).
//
// Aperture elements "stop the tracking for the particles found to be outside"
// (PAPER.md:178).  A stopped particle is frozen, so it can be retired: every compact_every
// turns the alive particles are packed to the front of a working SoA (stable partition:
// warp ballot + popc, block scan, tile offsets) so that the tracking kernel's warps stay
// full; each retired particle is written straight to its final place in the caller's
// arrays through its origin index.  HBM-bound, 2 x n x 112 B per pass.
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

// Pass 1: alive count per tile.
__global__ void __launch_bounds__(kTile) count_alive_kernel(const int64_t *__restrict__ state,
                                                            const int64_t *n_src_ptr, int64_t n_src_val,
                                                            int64_t *tile_counts) {
  const int64_t n_src = n_src_ptr ? *n_src_ptr : n_src_val;
  const int64_t i = static_cast<int64_t>(blockIdx.x) * kTile + threadIdx.x;
  const int alive = (i < n_src) && (state[i] == 1);
  const int cnt = __syncthreads_count(alive);
  if (threadIdx.x == 0) tile_counts[blockIdx.x] = cnt;
}

// Pass 2: exclusive scan of the tile counts in place (one CTA), total -> *n_dst.
__global__ void __launch_bounds__(1024) scan_tiles_kernel(int64_t *tile_counts, int64_t n_tiles, int64_t *n_dst) {
  __shared__ int64_t warp_sums[32];
  __shared__ int64_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int64_t start = 0; start < n_tiles; start += 1024) {
    const int64_t i = start + threadIdx.x;
    const int64_t v = (i < n_tiles) ? tile_counts[i] : 0;
    int64_t incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int64_t t = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl += t;
    }
    if (lane == 31) warp_sums[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      int64_t w = warp_sums[lane];
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const int64_t t = __shfl_up_sync(0xffffffffu, w, d);
        if (lane >= d) w += t;
      }
      warp_sums[lane] = w;  // inclusive over warps
    }
    __syncthreads();
    const int64_t before = carry + (warp ? warp_sums[warp - 1] : 0);
    if (i < n_tiles) tile_counts[i] = before + incl - v;
    __syncthreads();
    if (threadIdx.x == 0) carry += warp_sums[31];
    __syncthreads();
  }
  if (threadIdx.x == 0) *n_dst = carry;
}

// Pass 3: move.  Alive entries go to dst[tile_offset + rank]; lost entries of a working set
// retire to user[origin].
__global__ void __launch_bounds__(kTile) partition_move_kernel(xt_particles src, const int64_t *src_origin,
                                                               const int64_t *n_src_ptr, int64_t n_src_val,
                                                               const int64_t *tile_offsets, xt_particles dst,
                                                               int64_t *dst_origin, xt_particles user,
                                                               int retire_lost) {
  __shared__ int warp_counts[kTile / 32];
  const int64_t n_src = n_src_ptr ? *n_src_ptr : n_src_val;
  const int64_t i = static_cast<int64_t>(blockIdx.x) * kTile + threadIdx.x;
  if (static_cast<int64_t>(blockIdx.x) * kTile >= n_src) return;
  const bool in_range = i < n_src;
  const bool alive = in_range && (src.state[i] == 1);
  const unsigned ballot = __ballot_sync(0xffffffffu, alive);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) warp_counts[warp] = __popc(ballot);
  __syncthreads();
  int before = 0;
  for (int w = 0; w < warp; ++w) before += warp_counts[w];
  const int rank = before + __popc(ballot & ((1u << lane) - 1u));
  const int64_t origin = in_range ? (src_origin ? src_origin[i] : i) : 0;
  if (alive) {
    const int64_t j = tile_offsets[blockIdx.x] + rank;
    copy_particle(dst, j, src, i);
    dst_origin[j] = origin;
  } else if (in_range && retire_lost) {
    copy_particle(user, origin, src, i);
  }
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
    atomicAdd(&sh[b], 1u);
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
  plan.tile_counts = reinterpret_cast<int64_t *>(at);
  at += align256(static_cast<size_t>(plan.n_tiles) * 8);
  plan.n_active = reinterpret_cast<int64_t *>(at);
}

int launch_partition(const CompactPlan &plan, const xt_particles &src, const int64_t *src_origin,
                     bool src_is_user, int64_t n_part, const WorkSet &dst, const xt_particles &user,
                     cudaStream_t st) {
  if (n_part <= 0) return XT_OK;
  const unsigned grid = static_cast<unsigned>(plan.n_tiles);
  const int64_t *n_ptr = src_is_user ? nullptr : plan.n_active;
  count_alive_kernel<<<grid, kTile, 0, st>>>(src.state, n_ptr, n_part, plan.tile_counts);
  XT_CUDA(cudaGetLastError());
  // scan_tiles overwrites the counter with the new alive count, but the move kernel still
  // needs the old extent of src: keep it in the second counter slot.
  int64_t *n_old = plan.n_active + 1;
  if (!src_is_user) XT_CUDA(cudaMemcpyAsync(n_old, plan.n_active, 8, cudaMemcpyDeviceToDevice, st));
  scan_tiles_kernel<<<1, 1024, 0, st>>>(plan.tile_counts, plan.n_tiles, plan.n_active);
  XT_CUDA(cudaGetLastError());
  partition_move_kernel<<<grid, kTile, 0, st>>>(src, src_origin, src_is_user ? nullptr : n_old, n_part,
                                               plan.tile_counts, dst.p, dst.origin, user, src_is_user ? 0 : 1);
  XT_CUDA(cudaGetLastError());
  count_launch(3);
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
  if (grid > 148 * 8) grid = 148 * 8;
  histogram_kernel<<<static_cast<unsigned>(grid), 256, static_cast<size_t>(n_bins + 1) * 4, st>>>(
      at_turn, state, n, bin_width, static_cast<int>(n_bins), reinterpret_cast<unsigned long long *>(hist));
  XT_CUDA(cudaGetLastError());
  count_launch();
  return XT_OK;
}

}  // namespace xt
