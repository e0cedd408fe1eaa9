// The tracking kernel for sm_100a.
//
// "Xtrack ... assembles and compiles a C kernel ... able to track the entire beamline"
// (PAPER.md:74): here that kernel is hand-written.  One thread owns one particle and keeps
// its state in registers across all elements and turns; SoA FP64 loads/stores happen only at
// the start and end of the launch.  The lattice image is streamed chunk by chunk from L2
// into shared memory with 1-D TMA bulk copies (cp.async.bulk + mbarrier complete_tx),
// double-buffered; every thread of the CTA reads the same record, so each LDS.128 is a
// broadcast.  Element dispatch is a switch on a value all lanes share (warp-uniform).
// Multipoles are a complex Horner recurrence, fully unrolled per order.
//
// The arithmetic below is written as plain a*b + c expressions in the canonical order of
// the production build lets nvcc contract them into DFMA, the
// validation build (--fmad=false) does not and is then bit-identical to the oracle on
// cavity-free lattices (sqrt and 1/x are IEEE-correct in both: -prec-sqrt/-prec-div).
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

// Per-particle registers.
struct Part {
  double x, px, y, py, zeta, delta, ptau, rpp, rvv, s;
  double opd2, b, g, rv0v;  // cached functions of (delta, ptau), refreshed after a cavity
  int64_t at_element;
  bool alive;
};

__device__ __forceinline__ void refresh_cached(Part &q, double opd, double b, double t, double igam2) {
  q.opd2 = opd * opd;
  q.b = b;
  q.g = t * igam2;
  q.rv0v = b / opd;
}

// M2: complex Horner, coefficients stored highest order first as (c[n], s[n]) pairs.
template <int N>
__device__ __forceinline__ void horner(const double2 *__restrict__ cs, double x, double y, double &re,
                                       double &im) {
  double2 top = cs[0];
  re = top.x;
  im = top.y;
#pragma unroll
  for (int k = 1; k <= N; ++k) {
    const double2 c = cs[k];
    const double nre = re * x + (c.x - im * y);
    const double nim = re * y + (c.y + im * x);
    re = nre;
    im = nim;
  }
}

__device__ __forceinline__ void horner_dispatch(int order, const double2 *cs, double x, double y, double &re,
                                                double &im) {
  switch (order) {
#define XT_H(N) \
  case N:       \
    horner<N>(cs, x, y, re, im); \
    break;
    XT_H(0) XT_H(1) XT_H(2) XT_H(3) XT_H(4) XT_H(5) XT_H(6) XT_H(7) XT_H(8) XT_H(9) XT_H(10)
    XT_H(11) XT_H(12) XT_H(13) XT_H(14) XT_H(15) XT_H(16) XT_H(17) XT_H(18) XT_H(19)
#undef XT_H
    default:
      horner<20>(cs, x, y, re, im);
      break;
  }
}

__device__ __forceinline__ void lose(Part &q, uint32_t elem, const double *__restrict__ s_table) {
  q.alive = false;
  q.at_element = static_cast<int64_t>(elem);
  q.s = s_table[elem];
}

// Push the particle through every record of one staged chunk.
__device__ __forceinline__ void track_chunk(Part &q, const unsigned char *rp, const TrackArgs &a) {
  for (;;) {
    const RecHdr h = *reinterpret_cast<const RecHdr *>(rp);
    const uint32_t type = h.tag & 0xffu;
    if (type == TAG_END) break;
    const double2 *slots = reinterpret_cast<const double2 *>(rp + sizeof(RecHdr));
    switch (type) {
      case TAG_DRIFT: {
        // M1 exact drift, cancellation-free zeta (DESIGN.md section 5 "Drift")
        if (q.alive) {
          const double t1 = q.px * q.px;
          const double pxy2 = q.py * q.py + t1;
          const double pz = sqrt(q.opd2 - pxy2);
          const double s1 = pz + q.b;
          const double den = pz * s1;
          const double rr = 1.0 / den;
          const double lr = h.p0 * rr;
          const double lpz = lr * s1;
          q.x = q.px * lpz + q.x;
          q.y = q.py * lpz + q.y;
          q.zeta = (q.g - pxy2) * lr + q.zeta;
        }
        rp += 16;
        break;
      }
      case TAG_MULT: {
        const int order = static_cast<int>(h.tag >> 8);
        if (q.alive) {
          double re, im;
          horner_dispatch(order, slots, q.x, q.y, re, im);
          q.px = q.px - re;
          q.py = q.py + im;
        }
        rp += 32 + 16 * order;
        break;
      }
      case TAG_CMULT: {
        const int order = static_cast<int>(h.tag >> 8);
        if (q.alive) {
          const double hxl = h.p0;
          const double wf = slots[0].x;
          double re, im;
          horner_dispatch(order, slots + 1, q.x, q.y, re, im);
          q.px = q.px - re;
          q.py = q.py + im;
          q.px = hxl * q.delta + q.px;
          q.px = q.px - wf * q.x;
          q.zeta = q.zeta - (hxl * q.x) * q.rv0v;
        }
        rp += 48 + 16 * order;
        break;
      }
      case TAG_CAVITY: {
        if (q.alive) {
          const double2 kv = slots[0];  // (kz, vn)
          const double phase = h.p0 - kv.x * q.zeta;
          q.ptau = kv.y * sin(phase) + q.ptau;
          const double t = q.ptau * (q.ptau + a.tib);
          q.delta = t / (sqrt(t + 1.0) + 1.0);
          const double opd = 1.0 + q.delta;
          q.rpp = 1.0 / opd;
          const double b = 1.0 + a.beta0 * q.ptau;
          q.rvv = opd / b;
          refresh_cached(q, opd, b, t, a.igam2);
        }
        rp += 32;
        break;
      }
      case TAG_SROT: {
        if (q.alive) {
          const double2 cs = slots[0];  // (cos_z, sin_z)
          const double nx = cs.x * q.x + cs.y * q.y;
          const double ny = cs.x * q.y - cs.y * q.x;
          const double npx = cs.x * q.px + cs.y * q.py;
          const double npy = cs.x * q.py - cs.y * q.px;
          q.x = nx;
          q.y = ny;
          q.px = npx;
          q.py = npy;
        }
        rp += 32;
        break;
      }
      case TAG_SHIFT: {
        if (q.alive) {
          const double2 d = slots[0];
          q.x = q.x - d.x;
          q.y = q.y - d.y;
        }
        rp += 32;
        break;
      }
      case TAG_RECT: {
        if (q.alive) {
          const double2 xr = slots[0], yr = slots[1];
          const bool inside = (q.x >= xr.x) && (q.x <= xr.y) && (q.y >= yr.x) && (q.y <= yr.y);
          if (!inside) lose(q, h.elem, a.s_table);
        }
        rp += 48;
        break;
      }
      case TAG_ELLIPSE: {
        if (q.alive) {
          const double2 ba = slots[0];  // (b2, a2)
          const double tt = (q.x * q.x) * ba.x + (q.y * q.y) * ba.y;
          const bool inside = (tt <= h.p0);
          if (!inside) lose(q, h.elem, a.s_table);
        }
        rp += 32;
        break;
      }
      default:  // cannot happen: the packer emits only the tags above
        rp += 16;
        break;
    }
  }
}

__global__ void __launch_bounds__(512) xt_track_kernel(const TrackArgs a) {
  extern __shared__ __align__(128) unsigned char smem[];
  // smem layout: [0,16) two mbarriers; [128, 128+chunk_bytes) buffer 0; then buffer 1
  const uint32_t bar0 = smem_addr(smem);
  unsigned char *const buf0 = smem + 128;

  const int64_t n_active = a.n_active ? *a.n_active : a.n_part;
  const int64_t base = static_cast<int64_t>(blockIdx.x) * blockDim.x;
  if (base >= n_active) return;  // CTA-uniform
  const int64_t i = base + threadIdx.x;
  const bool valid = i < n_active;

  Part q;
  int64_t at_turn = 0;
  bool alive_at_load = false;
  q.alive = false;
  q.at_element = 0;
  q.s = 0.0;
  if (valid) {
    alive_at_load = (a.p.state[i] == 1);
  }
  if (alive_at_load) {
    q.x = a.p.x[i];
    q.px = a.p.px[i];
    q.y = a.p.y[i];
    q.py = a.p.py[i];
    q.zeta = a.p.zeta[i];
    q.delta = a.p.delta[i];
    q.ptau = a.p.ptau[i];
    q.rpp = a.p.rpp[i];
    q.rvv = a.p.rvv[i];
    q.s = a.p.s[i];
    at_turn = a.p.at_turn[i];
    q.at_element = a.p.at_element ? a.p.at_element[i] : 0;
    q.alive = true;
    const double opd = 1.0 + q.delta;
    const double b = 1.0 + a.beta0 * q.ptau;
    const double t = q.ptau * (q.ptau + a.tib);
    refresh_cached(q, opd, b, t, a.igam2);
  } else {
    q.x = q.px = q.y = q.py = q.zeta = q.delta = q.ptau = 0.0;
    q.rpp = q.rvv = 1.0;
    q.opd2 = q.b = q.rv0v = 1.0;
    q.g = 0.0;
  }

  const bool single = (a.n_chunks == 1);
  if (threadIdx.x == 0) {
    mbar_init(bar0, 1);
    mbar_init(bar0 + 8, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    const ChunkDesc d = a.chunks[0];
    tma_load_chunk(bar0, smem_addr(buf0), a.image + d.offset, d.nbytes);
  }

  if (single) {
    // Whole lattice resident in buffer 0: warps run free, no CTA-level synchronisation.
    mbar_wait(bar0, 0);
    for (int64_t turn = 0; turn < a.n_turns; ++turn) {
      if (!__any_sync(0xffffffffu, q.alive)) break;
      track_chunk(q, buf0, a);
      if (q.alive) at_turn += 1;
    }
  } else {
    const int64_t total = a.n_turns * a.n_chunks;
    int64_t gidx = 0;  // global chunk counter: buffer = gidx & 1, phase parity = (gidx >> 1) & 1
    int32_t c = 0;
    bool any = true;
    while (gidx < total) {
      if (threadIdx.x == 0 && gidx + 1 < total) {
        // buffer (gidx+1)&1 was released by the __syncthreads_or that ended iteration gidx-1
        const int32_t cn = (c + 1 == a.n_chunks) ? 0 : c + 1;
        const ChunkDesc d = a.chunks[cn];
        const uint32_t nb = static_cast<uint32_t>((gidx + 1) & 1);
        tma_load_chunk(bar0 + 8 * nb, smem_addr(buf0 + static_cast<size_t>(nb) * a.chunk_bytes),
                       a.image + d.offset, d.nbytes);
      }
      const uint32_t cb = static_cast<uint32_t>(gidx & 1);
      mbar_wait(bar0 + 8 * cb, static_cast<uint32_t>((gidx >> 1) & 1));
      if (__any_sync(0xffffffffu, q.alive)) track_chunk(q, buf0 + static_cast<size_t>(cb) * a.chunk_bytes, a);
      ++gidx;
      if (++c == a.n_chunks) {
        c = 0;
        if (q.alive) at_turn += 1;  // T: turn completed
      }
      any = __syncthreads_or(q.alive ? 1 : 0) != 0;
      if (!any) break;
    }
    if (!any && gidx < total) {
      // every particle of the CTA is lost: drain the copy still in flight before exiting
      mbar_wait(bar0 + 8 * static_cast<uint32_t>(gidx & 1), static_cast<uint32_t>((gidx >> 1) & 1));
    }
  }

  // W: store (only particles that were alive when the launch started can have changed)
  if (alive_at_load) {
    a.p.x[i] = q.x;
    a.p.px[i] = q.px;
    a.p.y[i] = q.y;
    a.p.py[i] = q.py;
    a.p.zeta[i] = q.zeta;
    a.p.delta[i] = q.delta;
    a.p.ptau[i] = q.ptau;
    a.p.rpp[i] = q.rpp;
    a.p.rvv[i] = q.rvv;
    a.p.s[i] = q.alive ? 0.0 : q.s;
    a.p.at_turn[i] = at_turn;
    a.p.state[i] = q.alive ? 1 : 0;
    if (a.p.at_element) a.p.at_element[i] = q.at_element;
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

}  // namespace

int launch_track(const xt_lattice *lat, const xt_particles &p, int64_t n_part, const int64_t *d_n_active,
                 int64_t n_turns, int block, cudaStream_t st) {
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
  a.beta0 = lat->k.beta0;
  a.tib = lat->k.tib;
  a.igam2 = lat->k.igam2;
  const size_t smem = 128 + (lat->info.n_chunks == 1 ? 1 : 2) * static_cast<size_t>(lat->info.chunk_bytes);
  static bool attr_set = false;
  if (!attr_set) {
    XT_CUDA(cudaFuncSetAttribute(xt_track_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 128 + 2 * 65536));
    attr_set = true;
  }
  const int64_t grid = (n_part + block - 1) / block;
  if (grid > 2147483647LL) {
    set_error("xt_track: too many particles for one launch");
    return XT_ERR_INVALID_ARG;
  }
  xt_track_kernel<<<static_cast<unsigned>(grid), block, smem, st>>>(a);
  count_launch();
  XT_CUDA(cudaGetLastError());
  return XT_OK;
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
