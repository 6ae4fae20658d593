// Host build of paper_2105_08026_b200/csrc/fastmath.cuh and philox.cuh::u01 for tests/test_fastmath_host.py.
// usage: fastmath_host <exp|expm1|log[2]|sqrt[2]|sqrt_both_root[2]|sqrt_both_inv[2]|sin2pi|cos2pi|u01|u32> (a trailing 2: the two-Newton-step variant) < binary doubles (u01: pairs of uint32 packed in uint64) > binary doubles
#include <cstdio>
#include <cstring>
#include <vector>
#include "../paper_2105_08026_b200/csrc/philox.cuh"
#include "../paper_2105_08026_b200/csrc/fastmath.cuh"

int main(int argc, char** argv) {
  if (argc < 2) return 2;
  std::vector<double> in;
  double buf[4096];
  size_t n;
  while ((n = fread(buf, sizeof(double), 4096, stdin)) > 0) in.insert(in.end(), buf, buf + n);
  std::vector<double> out(in.size());
  for (size_t i = 0; i < in.size(); ++i) {
    if (!strcmp(argv[1], "exp")) out[i] = hm::hm_exp_fast(in[i]);
    else if (!strcmp(argv[1], "log")) out[i] = hm::hm_log_pos_n<1>(in[i]);
    else if (!strcmp(argv[1], "log2")) out[i] = hm::hm_log_pos_n<2>(in[i]);
    else if (!strcmp(argv[1], "expm1")) out[i] = hm::hm_expm1_nonpos(in[i]);
    else if (!strcmp(argv[1], "sqrt")) out[i] = hm::hm_sqrt_fast_n<1>(in[i]);
    else if (!strcmp(argv[1], "sqrt2")) out[i] = hm::hm_sqrt_fast_n<2>(in[i]);
    else if (!strcmp(argv[1], "sqrt_both_root")) { double g, ig; hm::hm_sqrt_rsqrt_n<1>(in[i], &g, &ig); out[i] = g; }
    else if (!strcmp(argv[1], "sqrt_both_inv")) { double g, ig; hm::hm_sqrt_rsqrt_n<1>(in[i], &g, &ig); out[i] = ig; }
    else if (!strcmp(argv[1], "sqrt_both_root2")) { double g, ig; hm::hm_sqrt_rsqrt_n<2>(in[i], &g, &ig); out[i] = g; }
    else if (!strcmp(argv[1], "sqrt_both_inv2")) { double g, ig; hm::hm_sqrt_rsqrt_n<2>(in[i], &g, &ig); out[i] = ig; }
    else if (!strcmp(argv[1], "sin2pi")) { double sn, cs; hm::hm_sincos2pi(in[i], &sn, &cs); out[i] = sn; }
    else if (!strcmp(argv[1], "cos2pi")) { double sn, cs; hm::hm_sincos2pi(in[i], &sn, &cs); out[i] = cs; }
    else if (!strcmp(argv[1], "u01")) { uint64_t w; memcpy(&w, &in[i], 8); out[i] = hm::u01((uint32_t)(w >> 32), (uint32_t)w); }
    else if (!strcmp(argv[1], "u32")) { uint64_t w; memcpy(&w, &in[i], 8); out[i] = hm::u01_32((uint32_t)w); }
    else return 2;
  }
  fwrite(out.data(), sizeof(double), out.size(), stdout);
  return 0;
}
