// sanitize_main.cpp — driver that runs the oracle's event loop under AddressSanitizer / UBSan ("host oracle under
// -fsanitize=address,undefined").  TEST INFRASTRUCTURE like the rest of oracle/: built and run only by tests/test_oracle_sanitized.py,
// together with oracle.cpp, into a temporary directory.
//
//   oracle_san <process> <n_ext> <n_events> <in.bin> <out.bin>
//
// in.bin : double params_old[9], params_new[9], momenta[n_ext][4][n_events] (the SoA layout of orc_reweight), weights[n_events]
// out.bin: double me_old[n_events], me_new[n_events], w_new[n_events]
// Every buffer is a heap allocation of exactly the documented size, so a read or write past one of them is reported.
#include <cstdio>
#include <cstdlib>
#include <vector>

extern "C" int orc_reweight(const char* proc, const double* par_old, const double* par_new, const double* momenta, const double* weights,
                            double* me_old, double* me_new, double* w_new, long n_events, int nthreads);
extern "C" int orc_me2(const char* proc, const double* par, const double* p, double* out);

int main(int argc, char** argv) {
  if (argc != 6) { std::fprintf(stderr, "usage: oracle_san process n_ext n_events in.bin out.bin\n"); return 2; }
  const char* proc = argv[1];
  const long next = std::atol(argv[2]), n = std::atol(argv[3]);
  std::vector<double> po(9), pn(9), mom((size_t)next * 4 * n), w((size_t)n), a((size_t)n), b((size_t)n), o((size_t)n);
  std::FILE* f = std::fopen(argv[4], "rb");
  if (!f) return 3;
  bool ok = std::fread(po.data(), 8, 9, f) == 9 && std::fread(pn.data(), 8, 9, f) == 9 && std::fread(mom.data(), 8, mom.size(), f) == mom.size() &&
            std::fread(w.data(), 8, w.size(), f) == w.size();
  std::fclose(f);
  if (!ok) return 4;
  if (orc_reweight(proc, po.data(), pn.data(), mom.data(), w.data(), a.data(), b.data(), o.data(), n, 2) < 0) return 5;
  // the single-event entry point on a buffer of exactly n_ext * 4 doubles (event 0)
  std::vector<double> p((size_t)next * 4);
  for (long ip = 0; ip < next; ip++) for (int mu = 0; mu < 4; mu++) p[4 * ip + mu] = mom[(size_t)(ip * 4 + mu) * n];
  double one = 0.0;
  if (orc_me2(proc, po.data(), p.data(), &one) != 0 || !(one == a[0])) return 6;
  f = std::fopen(argv[5], "wb");
  if (!f) return 7;
  ok = std::fwrite(a.data(), 8, a.size(), f) == a.size() && std::fwrite(b.data(), 8, b.size(), f) == b.size() && std::fwrite(o.data(), 8, o.size(), f) == o.size();
  std::fclose(f);
  return ok ? 0 : 8;
}
