// Host-side emulation of ONE CTA of the register-resident 2-D FFT (paper_2505_14372_b200/csrc/fft_core.cuh).
// TEST HARNESS ONLY: it checks the index maps / exchange slots / in-register DFTs of the device code by running
// the __host__ __device__ phase functions for every thread id in sequence (barriers = loop boundaries).  It is
// never linked into the product library and is no CPU fallback: it transforms one field, from a file to a file.
//   usage: harness N in.bin out_fwd.bin out_roundtrip.bin   (N*N complex64 raster)
#include <cstdio>
#include <cstdlib>
#include <vector>
#include "../../paper_2505_14372_b200/csrc/fft_core.cuh"
using namespace ptk;

template <class G>
int run(const char* fin, const char* ffwd, const char* frt) {
  typedef Lay<G> L;
  const int N = G::N, T = G::T;
  std::vector<cf> in((size_t)N * N), out((size_t)N * N), rt((size_t)N * N);
  FILE* f = fopen(fin, "rb"); if (!f || fread(in.data(), sizeof(cf), in.size(), f) != in.size()) return 2; fclose(f);
  std::vector<cf> sm(L::XBUF), tw(L::TW);
  for (int i = 0; i < L::TW; ++i) L::fill_twiddle(tw.data(), i);
  struct Regs { cf r[32]; };
  std::vector<Regs> vv(T);
  auto v = [&](int t) -> cf (&)[32] { return vv[t].r; };
  // load in R-layout, and check the native-index inverse maps on the way
  for (int t = 0; t < T; ++t)
    for (int r = 0; r < 32; ++r) {
      int y = L::r_y(t, r), x = L::r_x(t, r);
      if (L::r_native_of(y, x) != L::native(t, r)) { printf("r_native_of mismatch\n"); return 3; }
      v(t)[r] = in[(size_t)y * N + x];
    }
  // ---- forward
  for (int t = 0; t < T; ++t) L::phase1_fwd(v(t), tw.data(), t);
  for (int t = 0; t < T; ++t) L::x1_store_p1(v(t), sm.data(), t);
  for (int t = 0; t < T; ++t) L::x1_load_p2(v(t), sm.data(), t);
  for (int t = 0; t < T; ++t) L::template phase2<-1>(v(t));
  for (int t = 0; t < T; ++t) L::x2_store_p2(v(t), sm.data(), t);
  for (int t = 0; t < T; ++t) L::x2_load_p3(v(t), sm.data(), t);
  for (int t = 0; t < T; ++t) L::template phase3<-1>(v(t));
  std::vector<int> seen((size_t)N * N, 0);
  for (int t = 0; t < T; ++t)
    for (int r = 0; r < 32; ++r) {
      int qy = L::f_qy(t, r), qx = L::f_qx(t, r);
      if (L::f_native_of(qy, qx) != L::native(t, r)) { printf("f_native_of mismatch\n"); return 3; }
      seen[(size_t)qy * N + qx]++;
      out[(size_t)qy * N + qx] = v(t)[r];
    }
  for (size_t i = 0; i < seen.size(); ++i) if (seen[i] != 1) { printf("F-layout not a bijection\n"); return 4; }
  // ---- inverse
  for (int t = 0; t < T; ++t) L::template phase3<+1>(v(t));
  for (int t = 0; t < T; ++t) L::x2_store_p3(v(t), sm.data(), t);
  for (int t = 0; t < T; ++t) L::x2_load_p2(v(t), sm.data(), t);
  for (int t = 0; t < T; ++t) L::template phase2<+1>(v(t));
  for (int t = 0; t < T; ++t) L::x1_store_p2(v(t), sm.data(), t);
  for (int t = 0; t < T; ++t) L::x1_load_p1(v(t), sm.data(), t);
  for (int t = 0; t < T; ++t) L::phase1_inv(v(t), tw.data(), t);
  for (int t = 0; t < T; ++t)
    for (int r = 0; r < 32; ++r) rt[(size_t)L::r_y(t, r) * N + L::r_x(t, r)] = v(t)[r];
  f = fopen(ffwd, "wb"); fwrite(out.data(), sizeof(cf), out.size(), f); fclose(f);
  f = fopen(frt, "wb"); fwrite(rt.data(), sizeof(cf), rt.size(), f); fclose(f);
  return 0;
}

int main(int argc, char** argv) {
  if (argc < 5) return 1;
  int N = atoi(argv[1]);
  if (N == 128) return run<Geo<128>>(argv[2], argv[3], argv[4]);
  if (N == 64) return run<Geo<64>>(argv[2], argv[3], argv[4]);
  return 1;
}
