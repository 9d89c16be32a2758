// Host build of the register transforms (csrc/fft_reg.cuh with MVD_HOST_TEST): the same straight-line
// butterflies the CUDA kernels inline, run on the CPU so that tests/test_fft_reg_host.py can check every
// length against a plain DFT.  Reads "N dir" then 2N floats from stdin, writes 2N floats.
#define MVD_HOST_TEST
#include "../../paper_1308_0730_b200/csrc/fft_reg.cuh"

#include <cstdio>
#include <vector>

using namespace mvd;

template <int N>
static void run(int dir, std::vector<float>& v) {
  float2 x[N];
  for (int i = 0; i < N; ++i) x[i] = make_float2(v[2 * i], v[2 * i + 1]);
  if (dir < 0) FftReg<N, -1>::run(x);
  else FftReg<N, 1>::run(x);
  for (int i = 0; i < N; ++i) { v[2 * i] = x[i].x; v[2 * i + 1] = x[i].y; }
}

#define CASE(N) case N: run<N>(dir, v); break;

int main() {
  int n, dir;
  while (std::scanf("%d %d", &n, &dir) == 2) {
    std::vector<float> v(2 * n);
    for (float& t : v) if (std::scanf("%f", &t) != 1) return 2;
    switch (n) {
      CASE(2) CASE(3) CASE(4) CASE(5) CASE(6) CASE(7) CASE(8) CASE(9) CASE(10) CASE(12) CASE(14) CASE(15) CASE(16)
      CASE(18) CASE(20) CASE(21) CASE(24) CASE(25) CASE(27) CASE(28) CASE(30) CASE(32) CASE(35) CASE(36)
      default: return 3;
    }
    for (float t : v) std::printf("%.9g ", t);
    std::printf("\n");
  }
  return 0;
}
