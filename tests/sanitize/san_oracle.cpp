// ASan / UBSan driver for the CPU oracle (oracle/xt_oracle.cpp).  usage: san_oracle file...
// Each file holds one packed lattice buffer (well formed or not): the oracle parses it, derives the
// reference particle and the s table, and tracks a handful of particles for three turns.  The exit code is 0
// unless a sanitizer aborts the process.  TEST INFRASTRUCTURE.
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>

extern "C" {
struct xo_particles {
  double *x, *px, *y, *py, *zeta, *delta, *ptau, *rpp, *rvv, *s;
  int64_t *at_turn, *state, *at_element;
  double *min_margin;
};
int xo_init_derived(const void *packed, size_t nbytes, const double *delta, double *ptau, double *rpp, double *rvv,
                    int64_t n);
int xo_reference(const void *packed, size_t nbytes, double *beta0, double *gamma0);
int64_t xo_s_table(const void *packed, size_t nbytes, double *out, int64_t cap);
int xo_track(const void *packed, size_t nbytes, const xo_particles *P, int64_t n_part, int64_t n_turns);
}

int main(int argc, char **argv) {
  for (int i = 1; i < argc; ++i) {
    std::vector<unsigned char> file;
    if (FILE *f = std::fopen(argv[i], "rb")) {
      unsigned char tmp[4096];
      size_t n;
      while ((n = std::fread(tmp, 1, sizeof tmp, f)) > 0) file.insert(file.end(), tmp, tmp + n);
      std::fclose(f);
    }
    unsigned char *buf = static_cast<unsigned char *>(std::malloc(file.size() ? file.size() : 1));
    for (size_t k = 0; k < file.size(); ++k) buf[k] = file[k];
    double b0 = 0, g0 = 0;
    const int rc_ref = xo_reference(buf, file.size(), &b0, &g0);
    const int64_t n_el = xo_s_table(buf, file.size(), nullptr, 0);
    std::vector<double> st(n_el > 0 ? n_el : 1);
    if (n_el > 0) xo_s_table(buf, file.size(), st.data(), n_el);
    constexpr int N = 7;
    std::vector<double> a[10];
    for (auto &v : a) v.assign(N, 0.0);
    for (int k = 0; k < N; ++k) {
      a[0][k] = 1e-4 * (k - 3);       // x
      a[1][k] = 1e-6 * (k - 2);       // px
      a[2][k] = -2e-4 * (k - 3);      // y
      a[3][k] = 2e-6 * (k - 4);       // py
      a[4][k] = 0.01 * (k - 3);       // zeta
      a[5][k] = 1e-4 * (k - 3);       // delta
    }
    a[0][N - 1] = 0.5;                // far outside any aperture
    std::vector<int64_t> at_turn(N, 0), state(N, 1), at_el(N, -1);
    std::vector<double> mm(N, 1e300);
    const int rc_init = xo_init_derived(buf, file.size(), a[5].data(), a[6].data(), a[7].data(), a[8].data(), N);
    xo_particles P{a[0].data(), a[1].data(), a[2].data(), a[3].data(), a[4].data(), a[5].data(), a[6].data(),
                   a[7].data(), a[8].data(), a[9].data(), at_turn.data(), state.data(), at_el.data(), mm.data()};
    const int rc = xo_track(buf, file.size(), &P, N, 3);
    int alive = 0;
    for (int k = 0; k < N; ++k) alive += state[k] == 1;
    std::printf("%s: reference rc %d, %lld elements, init rc %d, track rc %d, %d of %d alive\n", argv[i], rc_ref,
                (long long)n_el, rc_init, rc, alive, N);
    std::free(buf);
  }
  return 0;
}
