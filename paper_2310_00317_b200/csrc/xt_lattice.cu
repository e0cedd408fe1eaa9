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

// One record under construction: header + 16-byte slots of two doubles.
struct RecBuilder {
  std::vector<unsigned char> bytes;
  void header(uint32_t type, uint32_t order, uint32_t elem, double p0) {
    RecHdr h;
    h.tag = type | (order << 8);
    h.elem = elem;
    h.p0 = p0;
    bytes.resize(sizeof(RecHdr));
    std::memcpy(bytes.data(), &h, sizeof(RecHdr));
  }
  void slot(double a, double b) {
    const double v[2] = {a, b};
    const size_t at = bytes.size();
    bytes.resize(at + 16);
    std::memcpy(bytes.data() + at, v, 16);
  }
};

double inv_scale_factorial(int n) {  // n! as an exactly representable double (n <= 22)
  double f = 1.0;
  for (int i = 2; i <= n; ++i) f *= static_cast<double>(i);
  return f;
}

}  // namespace

int pack_image(const void *packed, size_t nbytes, uint32_t chunk_bytes, HostImage &out) {
  if (!packed) {
    set_error("xt_lattice_create: packed buffer is NULL");
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
  info.n_elements = n_elements;
  info.beta0 = beta0;
  info.gamma0 = gamma0;
  info.chunk_bytes = chunk_bytes;

  out.image.clear();
  out.chunks.clear();
  out.s_table.assign(n_elements, 0.0);

  const RecHdr end_rec{TAG_END | (static_cast<uint32_t>(sizeof(RecHdr)) << 16), 0u, 0.0};
  size_t chunk_start = 0;
  auto close_chunk = [&]() {
    const size_t at = out.image.size();
    out.image.resize(at + sizeof(RecHdr));
    std::memcpy(out.image.data() + at, &end_rec, sizeof(RecHdr));
    ChunkDesc d;
    d.offset = chunk_start;
    d.nbytes = static_cast<uint32_t>(out.image.size() - chunk_start);
    d.pad = 0;
    out.chunks.push_back(d);
    chunk_start = out.image.size();
  };
  auto append = [&](const RecBuilder &rb) {
    // keep room for the TAG_END record that closes the chunk
    if (out.image.size() - chunk_start + rb.bytes.size() + sizeof(RecHdr) > chunk_bytes) close_chunk();
    const size_t at = out.image.size();
    out.image.insert(out.image.end(), rb.bytes.begin(), rb.bytes.end());
    uint32_t tag;  // patch the record size into the upper half of the tag
    std::memcpy(&tag, out.image.data() + at, 4);
    tag |= static_cast<uint32_t>(rb.bytes.size()) << 16;
    std::memcpy(out.image.data() + at, &tag, 4);
    info.n_records += 1;
  };

  double s_pos = 0.0;
  RecBuilder rb;
  for (uint32_t ie = 0; ie < n_elements; ++ie) {
    const uint32_t type = r.get<uint32_t>();
    const uint32_t aux = r.get<uint32_t>();
    if (!r.ok) break;
    out.s_table[ie] = s_pos;
    if (type <= XT_LIMITELLIPSE) info.n_by_type[type] += 1;
    switch (type) {
      case XT_MARKER:
        break;  // no record: a marker is the identity map
      case XT_DRIFT: {
        const double length = r.real();
        rb.header(TAG_DRIFT, 0, ie, length);
        append(rb);
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
          const double f = inv_scale_factorial(n);
          cn[n] = knl[n] / f;
          sn[n] = ksl[n] / f;
        }
        if (hxl != 0.0) {
          // -k0l + hxl(1+delta) = -(k0l - hxl) + hxl*delta : fold the constant part into c[0]
          cn[0] = knl[0] - hxl;
          const double wf = (length != 0.0) ? (knl[0] * hxl) / length : 0.0;
          rb.header(TAG_CMULT, aux, ie, hxl);
          rb.slot(wf, 0.0);
          info.n_curved += 1;
        } else {
          rb.header(TAG_MULT, aux, ie, 0.0);
        }
        for (int n = order; n >= 0; --n) rb.slot(cn[n], sn[n]);  // Horner order: highest first
        append(rb);
        info.sum_order += order;
        break;
      }
      case XT_CAVITY: {
        const double volt = r.real();
        const double freq = r.real();
        const double lag_deg = r.real();
        const double lag_rad = lag_deg * (kPi / 180.0);
        const double kz = (2.0 * kPi * freq) / (beta0 * kClight);
        const double vn = (q0 * volt) / p0c;
        rb.header(TAG_CAVITY, 0, ie, lag_rad);
        rb.slot(kz, vn);
        append(rb);
        break;
      }
      case XT_SROTATION: {
        const double cz = r.real();
        const double sz = r.real();
        rb.header(TAG_SROT, 0, ie, 0.0);
        rb.slot(cz, sz);
        append(rb);
        break;
      }
      case XT_XYSHIFT: {
        const double dx = r.real();
        const double dy = r.real();
        rb.header(TAG_SHIFT, 0, ie, 0.0);
        rb.slot(dx, dy);
        append(rb);
        break;
      }
      case XT_LIMITRECT: {
        const double min_x = r.real();
        const double max_x = r.real();
        const double min_y = r.real();
        const double max_y = r.real();
        rb.header(TAG_RECT, 0, ie, 0.0);
        rb.slot(min_x, max_x);
        rb.slot(min_y, max_y);
        append(rb);
        info.has_aperture = 1;
        break;
      }
      case XT_LIMITELLIPSE: {
        const double a = r.real();
        const double b = r.real();
        const double a2 = a * a;
        const double b2 = b * b;
        rb.header(TAG_ELLIPSE, 0, ie, a2 * b2);
        rb.slot(b2, a2);
        append(rb);
        info.has_aperture = 1;
        break;
      }
      default:
        set_error("xt_lattice_create: unknown element type id");
        return XT_ERR_BAD_LATTICE;
    }
    if (!r.ok) break;
  }
  if (!r.ok) {
    set_error("xt_lattice_create: truncated buffer or non-finite parameter");
    return XT_ERR_BAD_LATTICE;
  }
  if (r.pos != nbytes) {
    set_error("xt_lattice_create: trailing bytes after the last element record");
    return XT_ERR_BAD_LATTICE;
  }
  close_chunk();  // also yields one END-only chunk for an empty / marker-only line
  info.n_chunks = static_cast<int64_t>(out.chunks.size());
  info.image_bytes = static_cast<int64_t>(out.image.size());
  info.circumference = s_pos;
  return XT_OK;
}

}  // namespace xt

// ------------------------------------------------------------------------------ C ABI
extern "C" int xt_lattice_create(const void *packed, size_t nbytes, xt_lattice **out) {
  if (!out) {
    xt::set_error("xt_lattice_create: out is NULL");
    return XT_ERR_INVALID_ARG;
  }
  xt::HostImage img;
  int rc = xt::pack_image(packed, nbytes, xt::kDefaultChunkBytes, img);
  if (rc != XT_OK) return rc;

  xt_lattice *lat = new (std::nothrow) xt_lattice;
  if (!lat) {
    xt::set_error("xt_lattice_create: host allocation failed");
    return XT_ERR_NOMEM;
  }
  lat->info = img.info;
  lat->k = img.k;
  lat->s_table_host = img.s_table;

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

extern "C" int64_t xt_lattice_s_table(const xt_lattice *lat, double *out, int64_t cap) {
  if (!lat || cap < 0 || (cap > 0 && !out)) {
    xt::set_error("xt_lattice_s_table: invalid argument");
    return XT_ERR_INVALID_ARG;
  }
  const int64_t n = static_cast<int64_t>(lat->s_table_host.size());
  for (int64_t i = 0; i < n && i < cap; ++i) out[i] = lat->s_table_host[i];
  return n;
}

extern "C" int64_t xt_lattice_pack_host(const void *packed, size_t nbytes, void *image, size_t cap,
                                        xt_lattice_info *info) {
  if (cap > 0 && !image) {
    xt::set_error("xt_lattice_pack_host: image is NULL but cap > 0");
    return XT_ERR_INVALID_ARG;
  }
  xt::HostImage img;
  const int rc = xt::pack_image(packed, nbytes, xt::kDefaultChunkBytes, img);
  if (rc != XT_OK) return rc;
  const size_t n = img.image.size() < cap ? img.image.size() : cap;
  if (n) std::memcpy(image, img.image.data(), n);
  if (info) *info = img.info;
  return static_cast<int64_t>(img.image.size());
}
