// Step P: the lattice packer.  Host code.  Turns the user's packed lattice
// buffer ("a sequence of ... objects ..., each corresponding to an accelerator element",
// PAPER.md:70) into the device image described in xt_internal.h and uploads it once.
//
// Constants are pre-computed here exactly as DESIGN.md section 5 prescribes (IEEE double,
// no FMA contraction: this file is built with -Xcompiler -ffp-contract=off), so that the
// kernel's arithmetic starts from the same FP64 values as the oracle's own parser:
//   c[n] = knl[n]/n!, s[n] = ksl[n]/n!;  curved: c[0] = knl[0] - hxl, wf = (knl[0]*hxl)/length
//   cavity: lag_rad = lag*(pi/180), kz = (2 pi f)/(beta0 c), vn = (q0 V)/p0c
//   ellipse: a2 = a*a, b2 = b*b, a2b2 = a2*b2
#include <cmath>
#include <cstring>
#include <new>

#include "xt_internal.h"

namespace xt {
namespace {

constexpr double kClight = 299792458.0;
constexpr double kPi = 3.14159265358979323846264338327950288;

struct Reader {
  const unsigned char *base;
  size_t size;
  size_t pos;
  bool ok = true;
  template <typename T>
  T get() {
    T v{};
    if (pos + sizeof(T) > size) {
      ok = false;
      return v;
    }
    std::memcpy(&v, base + pos, sizeof(T));
    pos += sizeof(T);
    return v;
  }
  double real() {  // a finite double or failure
    double v = get<double>();
    if (!std::isfinite(v)) ok = false;
    return v;
  }
};

// One record of the device image before serialisation.
struct Rec {
  uint32_t type = TAG_END;
  uint32_t order = 0;
  uint32_t flags = 0;  // TAG_PRE / TAG_POST / TAG_POST2 / TAG_MISAL
  uint32_t elem = 0;
  double p0 = 0.0;
  std::vector<double> slots;  // pairs, in the order the kernel reads them
  void slot(double a, double b) {
    slots.push_back(a);
    slots.push_back(b);
  }
  uint32_t bytes() const { return static_cast<uint32_t>(sizeof(RecHdr) + slots.size() * sizeof(double)); }
  uint32_t tag() const { return type | flags | (order << 8) | (bytes() << 16); }
};

double factorial(int n) {  // n! as an exactly representable double (n <= 22)
  double f = 1.0;
  for (int i = 2; i <= n; ++i) f *= static_cast<double>(i);
  return f;
}

}  // namespace

int pack_image(const void *packed, size_t nbytes, const PackOpts &opts, HostImage &out) {
  if (!packed) {
    set_error("xt_lattice_create: packed buffer is NULL");
    return XT_ERR_INVALID_ARG;
  }
  const uint32_t chunk_bytes = opts.chunk_bytes;
  if (chunk_bytes < 1024 || chunk_bytes > 65536 || (chunk_bytes % 128) != 0) {
    set_error("xt_lattice_create_ex: chunk_bytes must be a multiple of 128 in [1024, 65536]");
    return XT_ERR_INVALID_ARG;
  }
  Reader r{static_cast<const unsigned char *>(packed), nbytes, 0};
  if (nbytes < 48 || std::memcmp(r.base, "XTLAT001", 8) != 0) {
    set_error("xt_lattice_create: bad magic or buffer shorter than the 48-byte header");
    return XT_ERR_BAD_LATTICE;
  }
  r.pos = 8;
  const uint32_t version = r.get<uint32_t>();
  const uint32_t n_elements = r.get<uint32_t>();
  const double p0c = r.get<double>();
  const double mass0 = r.get<double>();
  const double q0 = r.get<double>();
  const uint64_t total = r.get<uint64_t>();
  if (version != 1 || total != nbytes) {
    set_error("xt_lattice_create: unsupported version or total_bytes does not match nbytes");
    return XT_ERR_BAD_LATTICE;
  }
  // every element record is at least 8 bytes (type, aux): a count the buffer cannot hold is rejected before
  // anything is sized from it (a 48-byte buffer announcing 2^32-1 elements must not allocate 32 GB)
  if (n_elements > (nbytes - 48) / 8 || n_elements >= (1u << 24)) {
    set_error("xt_lattice_create: n_elements does not fit the buffer (truncated) or exceeds 2^24 - 1");
    return XT_ERR_BAD_LATTICE;
  }
  if (!std::isfinite(p0c) || !std::isfinite(mass0) || !std::isfinite(q0) || !(p0c > 0.0) ||
      !(mass0 > 0.0)) {
    set_error("xt_lattice_create: p0c and mass0 must be finite and > 0, q0 finite");
    return XT_ERR_BAD_LATTICE;
  }

  // Reference particle (include/xt.h): E0 = sqrt(p0c^2 + mass0^2), beta0 = p0c/E0, gamma0 = E0/mass0
  const double e0 = std::sqrt(p0c * p0c + mass0 * mass0);
  const double beta0 = p0c / e0;
  const double gamma0 = e0 / mass0;
  out.k.beta0 = beta0;
  out.k.tib = 2.0 / beta0;
  out.k.igam2 = 1.0 / (gamma0 * gamma0);
  out.k.ib = 1.0 / beta0;
  out.k.ib2 = out.k.ib * out.k.ib;

  xt_lattice_info &info = out.info;
  info = xt_lattice_info{};
  out.extended = false;
  info.n_elements = n_elements;
  info.beta0 = beta0;
  info.gamma0 = gamma0;
  info.chunk_bytes = chunk_bytes;

  out.image.clear();
  out.chunks.clear();
  out.s_table.assign(n_elements, 0.0);
  out.mult_slot0.assign(n_elements, ~0ull);
  out.mult_wf_off.assign(n_elements, ~0ull);

  // ---- pass 1: one record per element (markers are the identity map: no record)
  std::vector<Rec> recs;
  recs.reserve(n_elements);
  double s_pos = 0.0;
  for (uint32_t ie = 0; ie < n_elements; ++ie) {
    const uint32_t type = r.get<uint32_t>();
    const uint32_t aux = r.get<uint32_t>();
    if (!r.ok) break;
    out.s_table[ie] = s_pos;
    if (type <= XT_LIMITELLIPSE) info.n_by_type[type] += 1;
    Rec rec;
    rec.elem = ie;
    switch (type) {
      case XT_MARKER:
        continue;
      case XT_DRIFT: {
        const double length = r.real();
        rec.type = TAG_DRIFT;
        rec.p0 = length;
        s_pos += length;
        break;
      }
      case XT_MULTIPOLE: {
        if (aux > XT_MAX_ORDER) {
          set_error("xt_lattice_create: multipole order exceeds XT_MAX_ORDER");
          return XT_ERR_BAD_LATTICE;
        }
        const int order = static_cast<int>(aux);
        const double hxl = r.real();
        const double length = r.real();
        double knl[XT_MAX_ORDER + 1], ksl[XT_MAX_ORDER + 1];
        for (int n = 0; n <= order; ++n) knl[n] = r.real();
        for (int n = 0; n <= order; ++n) ksl[n] = r.real();
        if (!r.ok) break;
        double cn[XT_MAX_ORDER + 1], sn[XT_MAX_ORDER + 1];
        for (int n = 0; n <= order; ++n) {
          const double f = factorial(n);
          cn[n] = knl[n] / f;
          sn[n] = ksl[n] / f;
        }
        rec.order = aux;
        if (hxl != 0.0) {
          // -k0l + hxl(1+delta) = -(k0l - hxl) + hxl*delta : fold the constant part into c[0]
          cn[0] = knl[0] - hxl;
          rec.type = TAG_CMULT;
          rec.p0 = hxl;
          info.n_curved += 1;
        } else {
          rec.type = TAG_MULT;
        }
        // two fixed slots in front, {l_pre, l_post} and {l_post2, wf} (the lengths are filled in by the
        // fusion pass), then the pairs in Horner order (highest first): every slot of the record sits
        // at an offset the handlers know at compile time
        rec.slot(0.0, 0.0);
        rec.slot(0.0, (hxl != 0.0 && length != 0.0) ? (knl[0] * hxl) / length : 0.0);
        for (int n = order; n >= 0; --n) rec.slot(cn[n], sn[n]);
        info.sum_order += order;
        break;
      }
      case XT_CAVITY: {
        const double volt = r.real();
        const double freq = r.real();
        const double lag_deg = r.real();
        rec.type = TAG_CAVITY;
        rec.p0 = lag_deg * (kPi / 180.0);                                    // lag_rad
        rec.slot((2.0 * kPi * freq) / (beta0 * kClight), (q0 * volt) / p0c);  // kz, vn
        break;
      }
      case XT_SROTATION: {
        const double cz = r.real();
        const double sz = r.real();
        rec.type = TAG_SROT;
        rec.slot(cz, sz);
        break;
      }
      case XT_XYSHIFT: {
        const double dx = r.real();
        const double dy = r.real();
        rec.type = TAG_SHIFT;
        rec.slot(dx, dy);
        break;
      }
      case XT_LIMITRECT: {
        const double min_x = r.real();
        const double max_x = r.real();
        const double min_y = r.real();
        const double max_y = r.real();
        rec.type = TAG_RECT;
        rec.slot(min_x, max_x);
        rec.slot(min_y, max_y);
        info.has_aperture = 1;
        break;
      }
      case XT_LIMITELLIPSE: {
        const double a = r.real();
        const double b = r.real();
        const double a2 = a * a;
        const double b2 = b * b;
        rec.type = TAG_ELLIPSE;
        rec.p0 = a2 * b2;
        rec.slot(b2, a2);
        info.has_aperture = 1;
        break;
      }
      case XT_QUADRUPOLE: {
        const double k1 = r.real();
        const double length = r.real();
        if (!r.ok) break;
        if (k1 == 0.0 || !(length > 0.0)) {
          set_error("xt_lattice_create: thick quadrupole needs k1 != 0 and length > 0 (a zero-strength one is a Drift)");
          return XT_ERR_BAD_LATTICE;
        }
        out.extended = true;
        rec.type = TAG_QUAD;
        rec.p0 = k1;
        rec.slot(length, 0.0);
        info.n_thick += 1;
        s_pos += length;
        break;
      }
      case XT_BEND: {
        const double k0 = r.real();
        const double h = r.real();
        const double length = r.real();
        if (!r.ok) break;
        if (!(k0 * h > 0.0) || !(length > 0.0)) {
          set_error("xt_lattice_create: thick bend needs k0*h > 0 and length > 0");
          return XT_ERR_BAD_LATTICE;
        }
        if (aux > 1u) {
          set_error("xt_lattice_create: thick bend model (aux) must be 0 ('expanded') or 1 ('full')");
          return XT_ERR_BAD_LATTICE;
        }
        out.extended = true;
        rec.type = aux == 1u ? TAG_BENDF : TAG_BEND;
        rec.p0 = k0;
        rec.slot(h, length);
        info.n_thick += 1;
        s_pos += length;
        break;
      }
      case XT_LIMITPOLYGON: {
        if (aux < 3 || aux > 256) {
          set_error("xt_lattice_create: a polygon aperture needs 3 to 256 vertices");
          return XT_ERR_BAD_LATTICE;
        }
        std::vector<double> vx(aux);
        for (uint32_t k = 0; k < aux; ++k) vx[k] = r.real();
        for (uint32_t k = 0; k < aux; ++k) rec.slot(vx[k], r.real());
        rec.type = TAG_POLY;
        info.has_aperture = 1;
        out.extended = true;
        break;
      }
      case XT_RADMULTIPOLE: {
        if (aux > XT_MAX_ORDER) {
          set_error("xt_lattice_create: multipole order exceeds XT_MAX_ORDER");
          return XT_ERR_BAD_LATTICE;
        }
        const int order = static_cast<int>(aux);
        const double hxl = r.real();
        const double length = r.real();
        double knl[XT_MAX_ORDER + 1], ksl[XT_MAX_ORDER + 1];
        for (int n = 0; n <= order; ++n) knl[n] = r.real();
        for (int n = 0; n <= order; ++n) ksl[n] = r.real();
        if (!r.ok) break;
        if (!(length > 0.0)) {
          set_error("xt_lattice_create: a radiating multipole needs length > 0");
          return XT_ERR_BAD_LATTICE;
        }
        rec.type = TAG_RMULT;
        rec.order = aux;
        rec.p0 = hxl;
        for (int n = order; n >= 1; --n) rec.slot(knl[n] / factorial(n), ksl[n] / factorial(n));
        rec.slot(knl[0] - hxl, ksl[0]);             // curvature folded into c[0] as in XT_MULTIPOLE (cancellation-free)
        rec.slot((knl[0] * hxl) / length, length);  // {wf, length}
        // (2/3) r0 (beta0 gamma0)^3, r0 = q0^2 e^2/(4 pi eps0 m c^2), e^2/(4 pi eps0) = 1.4399645478e-9 eV m
        const double r0 = ((q0 * q0) * 1.4399645478e-9) / mass0;
        const double bg0 = p0c / mass0;
        rec.slot(((2.0 / 3.0) * r0) * ((bg0 * bg0) * bg0), 0.0);
        out.extended = true;
        break;
      }
      case kMonitorType: {
        if (!opts.allow_monitor) {
          set_error("xt_lattice_create: unknown element type id");
          return XT_ERR_BAD_LATTICE;
        }
        rec.type = TAG_MON;
        rec.p0 = r.real();  // row
        out.extended = true;
        break;
      }
      default:
        set_error("xt_lattice_create: unknown element type id");
        return XT_ERR_BAD_LATTICE;
    }
    if (!r.ok) break;
    recs.push_back(std::move(rec));
  }
  if (!r.ok) {
    set_error("xt_lattice_create: truncated buffer or non-finite parameter");
    return XT_ERR_BAD_LATTICE;
  }
  if (r.pos != nbytes) {
    set_error("xt_lattice_create: trailing bytes after the last element record");
    return XT_ERR_BAD_LATTICE;
  }
  info.circumference = s_pos;

  // ---- pass 1b (production build only): consecutive drifts become ONE drift of the summed length.  px, py
  // and delta do not change in a drift, so D(l1) D(l2) = D(l1 + l2) exactly; what differs is one rounding
  // of x, y, zeta instead of two.  The validation build (--fmad=false) keeps every drift, as the oracle
  // does, and stays bit-identical to it.  Done before (and whether or not) records are fused, so that the
  // production results do not depend on the fusion option.
  info.n_drift_applies = info.n_by_type[XT_DRIFT];
#ifndef XT_FMAD_OFF
  if (opts.merge_drifts) {
    std::vector<Rec> merged;
    merged.reserve(recs.size());
    for (Rec &rec : recs) {
      if (rec.type == TAG_DRIFT && !merged.empty() && merged.back().type == TAG_DRIFT) {
        merged.back().p0 = merged.back().p0 + rec.p0;
        info.n_drift_applies -= 1;
      } else {
        merged.push_back(std::move(rec));
      }
    }
    recs.swap(merged);
  }
#endif

  // ---- pass 2: fuse.  A thin lattice is mostly drift - kick - drift, with
  // misaligned magnets wrapped in XYShift / SRotation.  A fused record applies
  // the same maps in the same order with the same arithmetic; what is shared is the dispatch
  // and, between consecutive drifts, the evaluation of what depends on (px, py) only.
  std::vector<Rec> fused;
  fused.reserve(recs.size());
  auto is = [&](size_t k, uint32_t type) { return k < recs.size() && recs[k].type == type; };
  auto is_mult = [&](size_t k) { return is(k, TAG_MULT) || is(k, TAG_CMULT); };
  for (size_t i = 0; i < recs.size();) {
    if (!opts.fuse) {
      fused.push_back(std::move(recs[i++]));
      continue;
    }
    if (is(i, TAG_DRIFT) && is(i + 1, TAG_DRIFT)) {  // two drifts in a row
      Rec d = std::move(recs[i]);
      d.flags |= TAG_POST;
      d.slot(recs[i + 1].p0, 0.0);
      fused.push_back(std::move(d));
      i += 2;
      continue;
    }
    size_t j = i;
    const bool pre = is(j, TAG_DRIFT);
    if (pre) ++j;
    const bool misal = is(j, TAG_SHIFT) && is(j + 1, TAG_SROT) && is_mult(j + 2) && is(j + 3, TAG_SROT) &&
                       is(j + 4, TAG_SHIFT);
    if (!misal && !is_mult(j)) {  // not a magnet group
      // half of a misalignment wrapper cut off from its magnet (by an aperture): still one dispatch
      if ((is(i, TAG_SHIFT) && is(i + 1, TAG_SROT)) || (is(i, TAG_SROT) && is(i + 1, TAG_SHIFT))) {
        Rec t = std::move(recs[i]);
        t.flags |= TAG_POST;
        t.slots.insert(t.slots.end(), recs[i + 1].slots.begin(), recs[i + 1].slots.end());
        fused.push_back(std::move(t));
        i += 2;
        continue;
      }
      fused.push_back(std::move(recs[i++]));
      continue;
    }
    const size_t m = misal ? j + 2 : j;
    size_t after = misal ? j + 5 : j + 1;
    Rec out_rec;
    out_rec.type = recs[m].type;
    out_rec.order = recs[m].order;
    out_rec.elem = recs[m].elem;
    out_rec.p0 = recs[m].p0;
    const bool post = is(after, TAG_DRIFT);
    const bool post2 = post && is(after + 1, TAG_DRIFT);
    if (pre) out_rec.flags |= TAG_PRE;
    if (post) out_rec.flags |= TAG_POST;
    if (post2) out_rec.flags |= TAG_POST2;
    if (misal) out_rec.flags |= TAG_MISAL;
    // slots: {l_pre, l_post} {l_post2, wf} [{dx, dy} {cos, sin} {cos', sin'} {dx', dy'}] pairs
    const std::vector<double> &ms = recs[m].slots;
    out_rec.slot(pre ? recs[i].p0 : 0.0, post ? recs[after].p0 : 0.0);
    out_rec.slot(post2 ? recs[after + 1].p0 : 0.0, ms[3]);
    if (misal) {
      for (size_t k : {j, j + 1, j + 3, j + 4})
        out_rec.slots.insert(out_rec.slots.end(), recs[k].slots.begin(), recs[k].slots.end());
    }
    out_rec.slots.insert(out_rec.slots.end(), ms.begin() + 4, ms.end());
    fused.push_back(std::move(out_rec));
    i = after + (post ? 1 : 0) + (post2 ? 1 : 0);
  }
  // ... and an elliptical aperture rides at the end of the multipole / drift record before it
  if (opts.fuse) {
    std::vector<Rec> merged;
    merged.reserve(fused.size());
    for (Rec &rec : fused) {
      const bool host = !merged.empty() && !(merged.back().flags & TAG_APER) &&
                        (merged.back().type == TAG_MULT || merged.back().type == TAG_CMULT ||
                         merged.back().type == TAG_DRIFT);
      if (rec.type == TAG_ELLIPSE && host) {
        Rec &m = merged.back();
        m.flags |= TAG_APER;
        m.slot(rec.slots[0], rec.slots[1]);                  // {b2, a2}
        m.slot(rec.p0, static_cast<double>(rec.elem));       // {a2 b2, element index}
      } else {
        merged.push_back(std::move(rec));
      }
    }
    fused.swap(merged);
  }
  info.n_records = static_cast<int64_t>(fused.size());
  {  // which instantiation of the tracking kernel suits the lattice: full of order-15 multipoles (errors on
     // every magnet), or of thin quadrupoles and sextupoles (orders 1 and 2)?
    int64_t n_mult = 0, n_15 = 0, n_low = 0;
    for (const Rec &rec : fused) {
      if (rec.type != TAG_MULT && rec.type != TAG_CMULT) continue;
      ++n_mult;
      if (rec.order == 15) ++n_15;
      if (rec.order == 1 || rec.order == 2) ++n_low;
    }
    out.fixed_order = 0;
    if (n_mult > 0 && 2 * n_15 >= n_mult) out.fixed_order = 15;
    else if (n_mult > 0 && 2 * n_low >= n_mult) out.fixed_order = 1 | (2 << 5);
  }
  for (const Rec &rec : fused) {
    if (rec.type == TAG_DRIFT) info.n_drift_evals += 1;
    if (rec.type == TAG_MULT || rec.type == TAG_CMULT)
      info.n_drift_evals += ((rec.flags & TAG_PRE) ? 1 : 0) + ((rec.flags & TAG_POST) ? 1 : 0);
  }

  // ---- pass 3: serialise.  Chunk = 16-byte preamble {tag of the first record} + records;
  // every record header carries the tag of the record that FOLLOWS it (TAG_END after the last
  // one of the chunk), so the kernel knows where it is going before it gets there.
  auto put_header = [&](size_t at, uint32_t next_tag, uint32_t elem, double p0) {
    RecHdr h;
    h.next = next_tag;
    h.elem = elem;
    h.p0 = p0;
    std::memcpy(out.image.data() + at, &h, sizeof(RecHdr));
  };
  size_t i = 0;
  do {
    const size_t chunk_start = out.image.size();
    out.image.resize(chunk_start + sizeof(RecHdr));
    size_t prev_hdr = chunk_start;  // where the next record's tag goes
    uint32_t prev_elem = 0;
    double prev_p0 = 0.0;
    while (i < fused.size()) {
      const Rec &rec = fused[i];
      const uint32_t nb = rec.bytes();
      if (sizeof(RecHdr) + nb > chunk_bytes) {
        set_error("xt_lattice_create_ex: chunk_bytes is smaller than one record");
        return XT_ERR_INVALID_ARG;
      }
      if (out.image.size() - chunk_start + nb > chunk_bytes) break;
      put_header(prev_hdr, rec.tag(), prev_elem, prev_p0);
      const size_t at = out.image.size();
      out.image.resize(at + nb);
      if (!rec.slots.empty())
        std::memcpy(out.image.data() + at + sizeof(RecHdr), rec.slots.data(), rec.slots.size() * sizeof(double));
      if (rec.type == TAG_MULT || rec.type == TAG_CMULT) {
        out.mult_wf_off[rec.elem] = at + sizeof(RecHdr) + 16 + 8;  // slot 1, second half
        out.mult_slot0[rec.elem] = at + sizeof(RecHdr) + 16 * (2 + ((rec.flags & TAG_MISAL) ? 4 : 0));
      }
      prev_hdr = at;
      prev_elem = rec.elem;
      prev_p0 = rec.p0;
      ++i;
    }
    put_header(prev_hdr, TAG_END, prev_elem, prev_p0);
    ChunkDesc d;
    d.offset = chunk_start;
    d.nbytes = static_cast<uint32_t>(out.image.size() - chunk_start);
    d.pad = 0;
    out.chunks.push_back(d);
  } while (i < fused.size());
  info.n_chunks = static_cast<int64_t>(out.chunks.size());
  info.image_bytes = static_cast<int64_t>(out.image.size());
  return XT_OK;
}

}  // namespace xt

// ------------------------------------------------------------------------------ C ABI
namespace xt {
namespace {
int resolve_pack_opts(const xt_lattice_opts *o, PackOpts &po) {
  po.chunk_bytes = kDefaultChunkBytes;
  po.fuse = true;
  if (!o) return XT_OK;
  if (o->chunk_bytes < 0 || o->fuse < 0 || o->fuse > 2) {
    set_error("xt_lattice_create_ex: chunk_bytes must be >= 0 and fuse one of 0 (default), 1 (on), 2 (off)");
    return XT_ERR_INVALID_ARG;
  }
  if (o->chunk_bytes > 0) po.chunk_bytes = static_cast<uint32_t>(o->chunk_bytes);
  if (o->fuse == 2) po.fuse = false;
  return XT_OK;
}
}  // namespace
}  // namespace xt

extern "C" int xt_lattice_create(const void *packed, size_t nbytes, xt_lattice **out) {
  return xt_lattice_create_ex(packed, nbytes, nullptr, out);
}

static int xt_lattice_create_ex_impl(const void *packed, size_t nbytes, const xt_lattice_opts *opts,
                                    xt_lattice **out) {
  if (!out) {
    xt::set_error("xt_lattice_create: out is NULL");
    return XT_ERR_INVALID_ARG;
  }
  xt::PackOpts po;
  const int rc = xt::resolve_pack_opts(opts, po);
  if (rc != XT_OK) return rc;
  return xt::create_lattice(packed, nbytes, po, out);
}

int xt::create_lattice(const void *packed, size_t nbytes, const PackOpts &po, xt_lattice **out) {
  xt::HostImage img;
  int rc = xt::pack_image(packed, nbytes, po, img);
  if (rc != XT_OK) return rc;

  xt_lattice *lat = new (std::nothrow) xt_lattice;
  if (!lat) {
    xt::set_error("xt_lattice_create: host allocation failed");
    return XT_ERR_NOMEM;
  }
  lat->info = img.info;
  lat->k = img.k;
  lat->s_table_host = img.s_table;
  lat->extended = img.extended;
  lat->mult_slot0 = img.mult_slot0;
  lat->mult_wf_off = img.mult_wf_off;
  lat->fixed_order = img.fixed_order;
  lat->packed_host.assign(static_cast<const unsigned char *>(packed), static_cast<const unsigned char *>(packed) + nbytes);

  auto fail = [&](cudaError_t e, const char *what) {
    int code = xt::cuda_fail(e, what);
    if (e == cudaErrorMemoryAllocation) code = XT_ERR_NOMEM;
    xt_lattice_destroy(lat);
    return code;
  };
  cudaError_t e = cudaGetDevice(&lat->device);
  if (e != cudaSuccess) return fail(e, "cudaGetDevice (no CUDA device? there is no CPU fallback)");
  if ((e = cudaDeviceGetAttribute(&lat->n_sm, cudaDevAttrMultiProcessorCount, lat->device)) != cudaSuccess)
    return fail(e, "cudaDeviceGetAttribute(multiProcessorCount)");
  const size_t n_s = img.s_table.empty() ? 1 : img.s_table.size();
  if ((e = cudaMalloc(&lat->d_image, img.image.size())) != cudaSuccess) return fail(e, "cudaMalloc(image)");
  if ((e = cudaMalloc(&lat->d_chunks, img.chunks.size() * sizeof(xt::ChunkDesc))) != cudaSuccess)
    return fail(e, "cudaMalloc(chunk table)");
  if ((e = cudaMalloc(&lat->d_s_table, n_s * sizeof(double))) != cudaSuccess) return fail(e, "cudaMalloc(s table)");
  if ((e = cudaMemcpy(lat->d_image, img.image.data(), img.image.size(), cudaMemcpyHostToDevice)) != cudaSuccess)
    return fail(e, "cudaMemcpy(image)");
  if ((e = cudaMemcpy(lat->d_chunks, img.chunks.data(), img.chunks.size() * sizeof(xt::ChunkDesc),
                      cudaMemcpyHostToDevice)) != cudaSuccess)
    return fail(e, "cudaMemcpy(chunk table)");
  if (!img.s_table.empty() &&
      (e = cudaMemcpy(lat->d_s_table, img.s_table.data(), img.s_table.size() * sizeof(double),
                      cudaMemcpyHostToDevice)) != cudaSuccess)
    return fail(e, "cudaMemcpy(s table)");
  *out = lat;
  return XT_OK;
}

extern "C" int xt_lattice_destroy(xt_lattice *lat) {
  if (!lat) return XT_OK;
  if (lat->d_image) cudaFree(lat->d_image);
  if (lat->d_chunks) cudaFree(lat->d_chunks);
  if (lat->d_s_table) cudaFree(lat->d_s_table);
  if (lat->d_knob_table) cudaFree(lat->d_knob_table);
  if (lat->d_knob_targets) cudaFree(lat->d_knob_targets);
  if (lat->d_knob_links) cudaFree(lat->d_knob_links);
  delete lat;
  return XT_OK;
}

extern "C" int xt_lattice_get_info(const xt_lattice *lat, xt_lattice_info *info) {
  if (!lat || !info) {
    xt::set_error("xt_lattice_get_info: NULL argument");
    return XT_ERR_INVALID_ARG;
  }
  *info = lat->info;
  return XT_OK;
}

static int64_t xt_lattice_s_table_impl(const xt_lattice *lat, double *out, int64_t cap) {
  if (!lat || cap < 0 || (cap > 0 && !out)) {
    xt::set_error("xt_lattice_s_table: invalid argument");
    return XT_ERR_INVALID_ARG;
  }
  const int64_t n = static_cast<int64_t>(lat->s_table_host.size());
  for (int64_t i = 0; i < n && i < cap; ++i) out[i] = lat->s_table_host[i];
  return n;
}

static int64_t xt_lattice_pack_host_impl(const void *packed, size_t nbytes, const xt_lattice_opts *opts,
                                        void *image, size_t cap, xt_lattice_info *info) {
  if (cap > 0 && !image) {
    xt::set_error("xt_lattice_pack_host: image is NULL but cap > 0");
    return XT_ERR_INVALID_ARG;
  }
  xt::PackOpts po;
  int rc = xt::resolve_pack_opts(opts, po);
  if (rc != XT_OK) return rc;
  xt::HostImage img;
  rc = xt::pack_image(packed, nbytes, po, img);
  if (rc != XT_OK) return rc;
  const size_t n = img.image.size() < cap ? img.image.size() : cap;
  if (n) std::memcpy(image, img.image.data(), n);
  if (info) *info = img.info;
  return static_cast<int64_t>(img.image.size());
}

// C ABI: no C++ exception may cross it (include/xt.h: "No exceptions, no abort()").  The bodies above use
// std::vector / std::map / std::string; a failed host allocation comes back as XT_ERR_NOMEM.
extern "C" int xt_lattice_create_ex(const void *packed, size_t nbytes, const xt_lattice_opts *opts, xt_lattice **out) {
  return xt::guarded<int>([&] { return xt_lattice_create_ex_impl(packed, nbytes, opts, out); });
}

extern "C" int64_t xt_lattice_pack_host(const void *packed, size_t nbytes, const xt_lattice_opts *opts, void *image, size_t cap, xt_lattice_info *info) {
  return xt::guarded<int64_t>([&] { return xt_lattice_pack_host_impl(packed, nbytes, opts, image, cap, info); });
}

extern "C" int64_t xt_lattice_s_table(const xt_lattice *lat, double *out, int64_t cap) {
  return xt::guarded<int64_t>([&] { return xt_lattice_s_table_impl(lat, out, cap); });
}
