// Test infrastructure only: runs the oracle's two entry points under
// -fsanitize=address,undefined on arrays read from raw files and prints a digest of every output, so that
// tests/test_oracle_pins.py can (a) see that the sanitizers stay silent and (b) compare the digest with the
// one the ordinary build gives. Built on demand by that test:
//   g++ -O1 -g -std=c++17 -fopenmp -fsanitize=address,undefined -fno-sanitize-recover=all \
//       oracle/sanitize_driver.cpp oracle/tpx3_oracle.cpp -o <tmp>/oracle_asan
// usage: oracle_asan <dir with x.u16 y.u16 toa.u64 tot.u16> W P wx wy wt
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <string>
#include <vector>

extern "C" int tpx3_oracle_run(uint64_t n, const uint16_t* x, const uint16_t* y, const uint64_t* toa, const uint16_t* tot,
                               uint64_t W, uint64_t P, int threads, uint32_t* perm, uint32_t* label, uint64_t* n_clusters,
                               uint32_t* c_label, uint32_t* c_size, uint32_t* c_shot, int64_t* c_sum_tot,
                               int64_t* c_sum_tot_x, int64_t* c_sum_tot_y, uint64_t* c_toa_peak, float* c_cx, float* c_cy,
                               int64_t* c_sum_tot_tof, float* c_ctof);
extern "C" int tpx3_oracle_localmax(uint64_t n, const uint16_t* x, const uint16_t* y, const uint64_t* toa,
                                    const uint16_t* tot, uint64_t wx, uint64_t wy, uint64_t wt, uint64_t P, int threads,
                                    uint32_t* perm, uint32_t* lmax, uint64_t* n_clusters, uint32_t* c_label,
                                    uint32_t* c_size, uint32_t* c_shot, int64_t* c_sum_tot, int64_t* c_sum_tot_x,
                                    int64_t* c_sum_tot_y, uint64_t* c_toa_peak, float* c_cx, float* c_cy,
                                    int64_t* c_sum_tot_tof, float* c_ctof);

template <class T>
static std::vector<T> slurp(const std::string& path) {
  FILE* f = fopen(path.c_str(), "rb");
  if (!f) { fprintf(stderr, "cannot open %s\n", path.c_str()); exit(2); }
  fseek(f, 0, SEEK_END);
  long bytes = ftell(f);
  fseek(f, 0, SEEK_SET);
  std::vector<T> v((size_t)bytes / sizeof(T));
  if (bytes && fread(v.data(), 1, (size_t)bytes, f) != (size_t)bytes) exit(2);
  fclose(f);
  return v;
}

static uint64_t fnv(uint64_t h, const void* p, size_t bytes) {
  const unsigned char* b = (const unsigned char*)p;
  for (size_t i = 0; i < bytes; ++i) { h ^= b[i]; h *= 1099511628211ull; }
  return h;
}

int main(int argc, char** argv) {
  if (argc != 8) return 2;
  const std::string dir = argv[1];
  const uint64_t W = strtoull(argv[2], 0, 10), P = strtoull(argv[3], 0, 10), wx = strtoull(argv[4], 0, 10),
                 wy = strtoull(argv[5], 0, 10), wt = strtoull(argv[6], 0, 10);
  const int threads = atoi(argv[7]);
  auto x = slurp<uint16_t>(dir + "/x.u16"), y = slurp<uint16_t>(dir + "/y.u16"), tot = slurp<uint16_t>(dir + "/tot.u16");
  auto toa = slurp<uint64_t>(dir + "/toa.u64");
  const uint64_t n = x.size();
  if (y.size() != n || tot.size() != n || toa.size() != n) return 2;
  for (int which = 0; which < 2; ++which) {
    std::vector<uint32_t> perm(n), label(n), cl(n), cs(n), csh(n);
    std::vector<int64_t> st(n), sx(n), sy(n), sf(n);
    std::vector<uint64_t> tp(n);
    std::vector<float> cx(n), cy(n), cf(n);
    uint64_t nc = 0;
    int rc = which == 0
                 ? tpx3_oracle_run(n, x.data(), y.data(), toa.data(), tot.data(), W, P, threads, perm.data(), label.data(),
                                   &nc, cl.data(), cs.data(), csh.data(), st.data(), sx.data(), sy.data(), tp.data(),
                                   cx.data(), cy.data(), sf.data(), cf.data())
                 : tpx3_oracle_localmax(n, x.data(), y.data(), toa.data(), tot.data(), wx, wy, wt, P, threads, perm.data(),
                                        label.data(), &nc, cl.data(), cs.data(), csh.data(), st.data(), sx.data(),
                                        sy.data(), tp.data(), cx.data(), cy.data(), sf.data(), cf.data());
    if (rc != 0) return 3;
    uint64_t h = 1469598103934665603ull;
    h = fnv(h, perm.data(), 4 * n); h = fnv(h, label.data(), 4 * n);
    h = fnv(h, cl.data(), 4 * nc); h = fnv(h, cs.data(), 4 * nc); h = fnv(h, csh.data(), 4 * nc);
    h = fnv(h, st.data(), 8 * nc); h = fnv(h, sx.data(), 8 * nc); h = fnv(h, sy.data(), 8 * nc);
    h = fnv(h, tp.data(), 8 * nc); h = fnv(h, cx.data(), 4 * nc); h = fnv(h, cy.data(), 4 * nc);
    h = fnv(h, sf.data(), 8 * nc); h = fnv(h, cf.data(), 4 * nc);
    printf("%s n=%llu hits=%llu digest=%016llx\n", which ? "localmax" : "run", (unsigned long long)n,
           (unsigned long long)nc, (unsigned long long)h);
  }
  return 0;
}
