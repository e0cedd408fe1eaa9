// ASan / UBSan driver for the HOST lattice packer (step P, csrc/xt_lattice.cu compiled as plain C++).
// usage: san_packer file...   each file holds one packed lattice buffer (well formed or not).
// Every buffer goes through xt_lattice_pack_host (size query, then fill) with the default options, with
// fusion off and with 1 KB chunks.  The exit code is 0 unless a sanitizer aborts the process; the
// packer's own verdict (bytes or error code) is printed per file.  TEST INFRASTRUCTURE.
#include <cstdio>
#include <cstdlib>
#include <string>
#include <vector>

#include "../../paper_2310_00317_b200/csrc/xt_internal.h"

namespace xt {  // what xt_api.cu provides in the library
static std::string g_err;
void set_error(const std::string &msg) { g_err = msg; }
int cuda_fail(cudaError_t, const char *what) {
  g_err = what;
  return XT_ERR_CUDA;
}
void count_launch(int64_t) {}
int check_device(const xt_lattice *, const char *) { return XT_ERR_CUDA; }
}  // namespace xt

static std::vector<unsigned char> slurp(const char *path) {
  std::vector<unsigned char> b;
  FILE *f = std::fopen(path, "rb");
  if (!f) return b;
  unsigned char tmp[4096];
  size_t n;
  while ((n = std::fread(tmp, 1, sizeof tmp, f)) > 0) b.insert(b.end(), tmp, tmp + n);
  std::fclose(f);
  return b;
}

int main(int argc, char **argv) {
  for (int i = 1; i < argc; ++i) {
    // an exactly-sized heap copy: any read past the end of the buffer is an ASan report
    const std::vector<unsigned char> file = slurp(argv[i]);
    unsigned char *buf = static_cast<unsigned char *>(std::malloc(file.size() ? file.size() : 1));
    for (size_t k = 0; k < file.size(); ++k) buf[k] = file[k];
    xt_lattice_opts variants[3] = {{0, 0, 0}, {0, 2, 0}, {1024, 0, 0}};
    for (const xt_lattice_opts &o : variants) {
      xt_lattice_info info{};
      const int64_t n = xt_lattice_pack_host(buf, file.size(), &o, nullptr, 0, &info);
      if (n > 0) {
        std::vector<unsigned char> img(static_cast<size_t>(n));
        const int64_t m = xt_lattice_pack_host(buf, file.size(), &o, img.data(), n, &info);
        std::printf("%s chunk=%lld fuse=%d: %lld bytes, %lld records\n", argv[i], (long long)o.chunk_bytes, o.fuse,
                    (long long)m, (long long)info.n_records);
      } else {
        std::printf("%s chunk=%lld fuse=%d: rc %lld\n", argv[i], (long long)o.chunk_bytes, o.fuse, (long long)n);
      }
    }
    std::free(buf);
  }
  return 0;
}
