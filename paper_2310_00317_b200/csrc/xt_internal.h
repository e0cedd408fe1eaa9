// Internal declarations shared by the translation units of libxt_b200 (never installed,
// never seen by the oracle).  Public contract: include/xt.h.
#pragma once

#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>
#include <new>
#include <string>
#include <vector>

#include "../../include/xt.h"

namespace xt {

// ------------------------------------------------------------------ device lattice image
// The image is a byte stream of 16-byte-aligned records, cut into chunks of at most
// chunk_bytes (one TMA bulk copy each).  A chunk is a 16-byte preamble followed by records.
// Preamble and every record start with a 16-byte header {u32 next; u32 elem; f64 p0}:
// `next` is the tag of the record that FOLLOWS (TAG_END after the last record of the chunk),
// so the kernel's dispatch never waits for the load of the record it is about to enter;
// elem and p0 belong to the record itself (unused in the preamble).
//
//   tag = type | flags | (order << 8) | (record bytes << 16)
//
// Fused records.  A multipole record may carry its neighbours: the drift before it
// (TAG_PRE), the XYShift + SRotation before and SRotation + XYShift after it (TAG_MISAL: a
// misaligned magnet), and one or two drifts after it (TAG_POST, + TAG_POST2).
// A drift record may carry a second drift (TAG_POST); an XYShift record the SRotation that
// follows it and vice versa (TAG_POST: second slot).  The maps are applied in element order
// with unchanged arithmetic; the dispatch is shared, and so is what two consecutive drifts
// would both compute from the unchanged (px, py).  Slots of a multipole record, in order:
//   {l_pre, l_post}; {l_post2, wf}   -- always present (zero where unused), so that every slot of the
//                                       record sits at an offset the handlers know at compile time;
//   {dx, dy}, {cos, sin}, {cos', sin'}, {dx', dy'} if MISAL;
//   the N+1 coefficient pairs (c[n], s[n]), n = N .. 0 (Horner order).
// The kernel loads the first four slots behind every header before the dispatch resolves: the extras
// and, without misalignment, the two leading pairs.
// In the production build consecutive drifts reach the fusion pass already merged into one drift of the
// summed length (xt_lattice.cu pass 1b), so TAG_POST2 only occurs in the validation build.
// A multipole or drift record may also end with the LimitEllipse that follows it (TAG_APER):
// its last two slots are then {b2, a2}, {a2*b2, element index of the aperture}.
// Unfused records:
//
//   TAG_DRIFT    p0 = length; {l_2nd, 0} with TAG_POST                           16 B (32 B)
//   TAG_MULT     p0 unused; two extras slots; (c[n], s[n]) pairs, n = N .. 0     48 + 16(N+1)
//   TAG_CMULT    p0 = hxl;  as above with c[0] = knl[0] - hxl and wf in the extras 48 + 16(N+1)
//   TAG_CAVITY   p0 = lag_rad; {kz, vn}                                          32 B
//   TAG_SROT     p0 unused; {cos_z, sin_z}                                       32 B
//   TAG_SHIFT    p0 unused; {dx, dy}                                             32 B
//   TAG_RECT     p0 unused; {min_x, max_x}; {min_y, max_y}                       48 B
//   TAG_ELLIPSE  p0 = a2*b2; {b2, a2}                                            32 B
//   TAG_QUAD     p0 = k1; {length, 0}   (thick quadrupole; never fused)          32 B
//   TAG_BEND     p0 = k0; {h, length}   (thick sector bend; never fused)         32 B
//   TAG_POLY     p0 unused; n vertices {x_k, y_k} (polygon aperture; never fused)  16 + 16 n
//
// elem = index of the element in the user's packed buffer (for a fused record: the
// multipole's; only aperture records ever report it).
enum : uint32_t {
  TAG_END = 0,
  TAG_DRIFT = 1,
  TAG_MULT = 2,
  TAG_CAVITY = 3,
  TAG_SROT = 4,
  TAG_SHIFT = 5,
  TAG_RECT = 6,
  TAG_ELLIPSE = 7,
  TAG_CMULT = 8,
  TAG_QUAD = 9,
  TAG_BEND = 10,
  TAG_POLY = 11,
  TAG_RMULT = 13,  // radiating multipole: p0 = hxl; (c[n], s[n]) pairs n = N .. 0 (c[0] = knl[0] - hxl); {wf, length}; {krad, 0}
  TAG_BENDF = 14,  // thick sector bend, 'full' map
  TAG_MON = 12,  // internal: store the coordinates of every alive particle into row p0 of the monitor buffer
  TAG_TYPE_MASK = 0xf,
  TAG_PRE = 0x10,   // a drift of length l_pre comes first
  TAG_POST = 0x20,  // a drift of length l_post follows the kick
  TAG_POST2 = 0x40,  // ... and a second one of length l_post2 (only with TAG_POST)
  TAG_MISAL = 0x80,  // shift + rotation before the kick, rotation + shift after it
  TAG_APER = 0x8000  // (top bit of the order byte) a LimitEllipse follows the record's last map
};

struct alignas(16) RecHdr {
  uint32_t next;
  uint32_t elem;
  double p0;
};
static_assert(sizeof(RecHdr) == 16, "record header must be one 16-byte slot");

struct alignas(16) ChunkDesc {
  uint64_t offset;  // byte offset into the image (multiple of 16)
  uint32_t nbytes;  // multiple of 16, <= chunk_bytes: preamble + records (there is no END record: TAG_END is the
                    // `next` field of the chunk's last header).  The kernel's slot prefetch and the run-time Horner
                    // loop read up to 64 bytes past the last record of a stage; the values are never used.  Behind
                    // the last buffer that is the 64 spare bytes of the allocation; behind buffer 0 it is the head
                    // of buffer 1, possibly while a bulk copy is writing it -- a read whose result is discarded.
  uint32_t pad;
};

struct RefConsts {
  double beta0;  // p0c / E0
  double tib;    // 2 / beta0
  double igam2;  // 1 / gamma0^2
  double ib;     // 1 / beta0
  double ib2;    // ib * ib
};

constexpr uint32_t kDefaultChunkBytes = 8192;

}  // namespace xt

struct xt_lattice {
  xt_lattice_info info{};
  xt::RefConsts k{};
  int device = -1;
  int n_sm = 0;  // multiprocessors of `device`: the grid quantum of the tracking kernel
  std::vector<double> s_table_host;
  std::vector<unsigned char> packed_host;  // the buffer the lattice was created from (xt_refine.cu re-reads it)
  bool extended = false;                   // thick maps or polygon apertures: the THICK kernels
  int fixed_order = 0;                     // which orders have unrolled handlers: 15 (most multipoles of order 15),
                                           // 1 | 2 << 5 (most of order 1 or 2), else 0
  std::vector<uint64_t> mult_slot0;        // per element: image offset of a multipole's first coefficient pair
  std::vector<uint64_t> mult_wf_off;       // per element: image offset of a multipole's weak-focusing term
  // time functions (xt_knobs.cu); all device memory, owned
  double *d_knob_table = nullptr;
  void *d_knob_targets = nullptr;
  void *d_knob_links = nullptr;
  int64_t n_knob_targets = 0, n_knob_steps = 0;
  unsigned char *d_image = nullptr;
  xt::ChunkDesc *d_chunks = nullptr;
  double *d_s_table = nullptr;
  double *d_monitor_rows = nullptr;  // not owned: where the TAG_MON records of an internal monitor line store
};

namespace xt {

// xt_api.cu
void set_error(const std::string &msg);
int cuda_fail(cudaError_t e, const char *what);
void count_launch(int64_t n = 1);
// XT_ERR_INVALID_ARG unless the current CUDA device is the one the lattice's image lives on (every entry
// point that takes a lattice checks this before it allocates or launches anything).
int check_device(const xt_lattice *lat, const char *fn);
// Runs the body of a C-ABI entry point; turns any C++ exception into an error code (the message is short
// enough for std::string's in-place buffer: reporting must not allocate).
template <class R, class F>
R guarded(F &&body) noexcept {
  try {
    return body();
  } catch (const std::bad_alloc &) {
    try { set_error("out of memory"); } catch (...) {}
    return static_cast<R>(XT_ERR_NOMEM);
  } catch (...) {
    try { set_error("C++ exception"); } catch (...) {}
    return static_cast<R>(XT_ERR_NOMEM);
  }
}
#define XT_CUDA(call)                                      \
  do {                                                     \
    cudaError_t e__ = (call);                              \
    if (e__ != cudaSuccess) return xt::cuda_fail(e__, #call); \
  } while (0)

// xt_lattice.cu: host packer (step P).  Builds the image bytes, chunk table, s table.
struct HostImage {
  std::vector<unsigned char> image;
  std::vector<ChunkDesc> chunks;
  std::vector<double> s_table;
  xt_lattice_info info{};
  RefConsts k{};
  bool extended = false;
  int fixed_order = 0;  // see xt_lattice::fixed_order
  std::vector<uint64_t> mult_slot0;   // per element: offset of a multipole's first coefficient pair (else ~0)
  std::vector<uint64_t> mult_wf_off;  // per element: offset of a multipole's weak-focusing term wf (else ~0)
};
struct PackOpts {
  uint32_t chunk_bytes = kDefaultChunkBytes;
  bool fuse = true;
  bool merge_drifts = true;    // production build: consecutive drifts -> one drift of the summed length (pass 1b)
  bool allow_monitor = false;  // accept the internal element type kMonitorType (xt_twiss4d_line builds such lines)
};
constexpr uint32_t kMonitorType = 11;  // packed-buffer type id, internal: {row} -> TAG_MON record
int create_lattice(const void *packed, size_t nbytes, const PackOpts &po, xt_lattice **out);
int pack_image(const void *packed, size_t nbytes, const PackOpts &opts, HostImage &out);

// xt_track.cu
// block: threads per CTA; ppt: particles per thread (1, 2, 3 or 4; 4 needs block <= 256); cold_in_regs: the
// per-particle functions of (delta, ptau) in registers instead of shared memory (ppt 2 or 3 only).
// TAG_MON records store into lat->d_monitor_rows (rows of n_part x 6 doubles: x, px, y, py, zeta, delta).
// queue: device scratch of balance_scratch_bytes() for the balanced mode (persistent CTAs drawing
// (group, block of turns) items from a ticket counter; cold_in_regs shapes without a device counter only),
// or nullptr.  balance: xt_track_opts.balance (< 0 never, 0 auto, 1 always, n > 1 always with n turns per item).
int launch_track(const xt_lattice *lat, const xt_particles &p, int64_t n_part,
                 const int64_t *d_n_active, int64_t n_turns, int block, int ppt, bool cold_in_regs,
                 cudaStream_t st, unsigned int *queue = nullptr, int balance = 0);
size_t balance_scratch_bytes(int64_t n_part, int block, int ppt);
// turns per item of the balanced mode for a launch of n_turns turns, and whether the auto rule would use it
int64_t balance_block_turns(const xt_lattice *lat, int64_t n_turns, int balance);
bool balance_pays(const xt_lattice *lat, int64_t n_turns, int balance);
int launch_init_derived(const xt_lattice *lat, const xt_particles &p, int64_t n, cudaStream_t st);

// xt_compact.cu (step C) -- SoA working set with an origin index
struct WorkSet {
  xt_particles p{};            // 10 f64 + at_turn, state, at_element (particle_id unused)
  int64_t *origin = nullptr;   // index in the caller's arrays
};
size_t compaction_workspace_bytes(int64_t n_part);
// Carves two WorkSets + counters + tile scratch out of `ws` (256-byte aligned pieces).
struct CompactPlan {
  WorkSet w[2];
  int64_t *n_active = nullptr;   // device counter holding the extent of the current working set
  int64_t *counter[2] = {nullptr, nullptr};  // n_active alternates between the two (a pass reads one, writes the other)
  unsigned long long *status = nullptr;      // per-tile status words of the single-pass scan
  unsigned int *ticket = nullptr;            // tile ticket counter
  uint32_t epoch = 0;                        // pass number of this call (tags the status words)
  int64_t n_tiles = 0;
};
void plan_compaction(void *ws, int64_t n_part, CompactPlan &plan);
// dst <- alive entries of src (stable); lost entries of src are written to `user` at their
// origin unless src_is_user.  The extent of src is read from plan.n_active unless src_is_user (then n_part);
// afterwards plan.n_active points to the counter that holds the new alive count.
int launch_partition(CompactPlan &plan, const xt_particles &src, const int64_t *src_origin,
                     bool src_is_user, int64_t n_part, const WorkSet &dst, const xt_particles &user,
                     cudaStream_t st);
int launch_scatter_back(const CompactPlan &plan, const WorkSet &src, int64_t n_part,
                        const xt_particles &user, cudaStream_t st);
int launch_histogram(const int64_t *at_turn, const int64_t *state, int64_t n, int64_t bin_width,
                     int64_t n_bins, int64_t *hist, cudaStream_t st);

// xt_peak.cu
int run_fma_peak(double *flops_per_s, double *ms, int pattern, cudaStream_t st);
int fma_peak_sweep_size();
int run_fma_peak_shape(int i, double *flops_per_s, double *ms, int *desc, cudaStream_t st);

}  // namespace xt
