// The user's packed lattice buffer (include/xt.h) re-read as a list of elements: what the host-side
// features beyond the hot path (xt_refine.cu, xt_knobs.cu) work from.  The buffer was validated by
// xt_lattice_create, which keeps a copy (xt_lattice::packed_host).
#pragma once
#include <cstdint>
#include <cstring>
#include <vector>

#include "../../include/xt.h"

namespace xt {

struct Elem {
  uint32_t type = 0, aux = 0;
  std::vector<double> v;  // parameters as stored in the packed buffer
  double length() const {
    if (type == XT_DRIFT) return v[0];
    if (type == XT_QUADRUPOLE) return v[1];
    if (type == XT_BEND) return v[2];
    return 0.0;
  }
  bool is_aperture() const { return type == XT_LIMITRECT || type == XT_LIMITELLIPSE || type == XT_LIMITPOLYGON; }
  bool is_any_aperture() const { return is_aperture(); }
};

// number of doubles behind the 8-byte element header (include/xt.h, element table)
inline int n_params(uint32_t type, uint32_t aux) {
  switch (type) {
    case XT_MARKER: return 0;
    case XT_DRIFT: return 1;
    case XT_MULTIPOLE: case XT_RADMULTIPOLE: return 2 + 2 * (static_cast<int>(aux) + 1);
    case XT_CAVITY: return 3;
    case XT_SROTATION: case XT_XYSHIFT: case XT_LIMITELLIPSE: case XT_QUADRUPOLE: return 2;
    case XT_LIMITRECT: return 4;
    case XT_BEND: return 3;
    case XT_LIMITPOLYGON: return 2 * static_cast<int>(aux);
    default: return -1;
  }
}

struct Line {
  double p0c = 0, mass0 = 0, q0 = 0;
  std::vector<Elem> el;
};

inline bool read_line(const std::vector<unsigned char> &buf, Line &line) {
  if (buf.size() < 48) return false;
  uint32_t n_el;
  std::memcpy(&n_el, buf.data() + 12, 4);
  std::memcpy(&line.p0c, buf.data() + 16, 8);
  std::memcpy(&line.mass0, buf.data() + 24, 8);
  std::memcpy(&line.q0, buf.data() + 32, 8);
  size_t off = 48;
  line.el.resize(n_el);
  for (uint32_t i = 0; i < n_el; ++i) {
    Elem &e = line.el[i];
    if (off + 8 > buf.size()) return false;
    std::memcpy(&e.type, buf.data() + off, 4);
    std::memcpy(&e.aux, buf.data() + off + 4, 4);
    off += 8;
    const int n = n_params(e.type, e.aux);
    if (n < 0 || off + 8 * static_cast<size_t>(n) > buf.size()) return false;
    e.v.resize(n);
    if (n) std::memcpy(e.v.data(), buf.data() + off, 8 * static_cast<size_t>(n));
    off += 8 * static_cast<size_t>(n);
  }
  return true;
}

// A packed lattice buffer (include/xt.h) under construction.
struct Writer {
  std::vector<unsigned char> b;
  uint32_t n = 0;
  explicit Writer(const Line &l) : b(48, 0) {
    std::memcpy(b.data(), "XTLAT001", 8);
    const uint32_t version = 1;
    std::memcpy(b.data() + 8, &version, 4);
    std::memcpy(b.data() + 16, &l.p0c, 8);
    std::memcpy(b.data() + 24, &l.mass0, 8);
    std::memcpy(b.data() + 32, &l.q0, 8);
  }
  void put(uint32_t type, uint32_t aux, const double *v, size_t nv) {
    const size_t at = b.size();
    b.resize(at + 8 + 8 * nv);
    std::memcpy(b.data() + at, &type, 4);
    std::memcpy(b.data() + at + 4, &aux, 4);
    if (nv) std::memcpy(b.data() + at + 8, v, 8 * nv);
    ++n;
  }
  void put(const Elem &e) { put(e.type, e.aux, e.v.data(), e.v.size()); }
  const std::vector<unsigned char> &finish() {
    const uint64_t total = b.size();
    std::memcpy(b.data() + 12, &n, 4);
    std::memcpy(b.data() + 40, &total, 8);
    return b;
  }
};

}  // namespace xt
