// fft_core.cuh — register-resident 2-D complex FFT of an N x N field held by one CTA (N = 64, 128).
//
// A field of N*N complex64 lives in the REGISTERS of T = N*N/32 threads, 32 elements per thread.  One 2-D
// FFT is three in-register phases joined by two shared-memory exchanges (the minimum for 2^14 points at 2^5
// per thread):
//
//   R-layout (real space)  thread (a, b), reg (n1y, n1x):  x = a + N2X*n1x,  y = b + N2Y*n1y
//     phase 1: DFT-N1X over n1x and DFT-N1Y over n1y, then twiddles W_N^(a*k1x) W_N^(b*k1y)
//   exchange X1 (warp-local 32x32 transpose: lane <-> register)
//     phase 2: DFT-N2X over a  (LP2 lines per thread)           -> qx = k1x + N1X*k2x
//   exchange X2 (CTA-wide: for each k1y a [b] x [qx] transpose)
//     phase 3: DFT-N2Y over b  (LP3 lines per thread)           -> qy = k1y + N1Y*k2y
//   F-layout (Fourier space) thread (qx, c), reg (ksel, k2y): k1y = c*LP3 + ksel, qy = k1y + N1Y*k2y
//
// The inverse runs the same phases backwards (conjugated constants), so no bit reversal is ever
// materialised: pointwise operators are indexed through the layout maps below.  Both exchanges use
// padded/skewed slots whose addresses are thread-base + compile-time immediates and are bank-conflict free
// for 8-byte accesses in both directions.
//
// Everything here is __host__ __device__ so that tests/test_fft_layout.py can emulate one CTA on the host
// (index maps only; the host build is a test harness, never a product path).
#pragma once
#include <cuda_runtime.h>

#if defined(__CUDACC__)
#define PTK_HD __host__ __device__ __forceinline__
#else
#define PTK_HD inline
#endif

namespace ptk {

typedef float2 cf;

PTK_HD cf cmul(cf a, cf b) { return make_float2(fmaf(-a.y, b.y, a.x * b.x), fmaf(a.y, b.x, a.x * b.y)); }
PTK_HD cf cmulc(cf a, cf b) { /* a * conj(b) */ return make_float2(fmaf(a.y, b.y, a.x * b.x), fmaf(a.y, b.x, -(a.x * b.y))); }
PTK_HD cf cadd(cf a, cf b) { return make_float2(a.x + b.x, a.y + b.y); }
PTK_HD cf csub(cf a, cf b) { return make_float2(a.x - b.x, a.y - b.y); }
PTK_HD cf cconj(cf a) { return make_float2(a.x, -a.y); }
PTK_HD cf cscale(cf a, float s) { return make_float2(a.x * s, a.y * s); }

// cos / sin (2 pi m / 32), correctly rounded float literals
PTK_HD constexpr float c32(int m) {
  switch (m & 31) {
    case 0: return 1.0f; case 1: return 0.98078525066375732f; case 2: return 0.92387950420379639f;
    case 3: return 0.83146959543228149f; case 4: return 0.70710676908493042f; case 5: return 0.55557024478912354f;
    case 6: return 0.38268342614173889f; case 7: return 0.19509032368659973f; case 8: return 0.0f;
    case 9: return -0.19509032368659973f; case 10: return -0.38268342614173889f; case 11: return -0.55557024478912354f;
    case 12: return -0.70710676908493042f; case 13: return -0.83146959543228149f; case 14: return -0.92387950420379639f;
    case 15: return -0.98078525066375732f; case 16: return -1.0f; case 17: return -0.98078525066375732f;
    case 18: return -0.92387950420379639f; case 19: return -0.83146959543228149f; case 20: return -0.70710676908493042f;
    case 21: return -0.55557024478912354f; case 22: return -0.38268342614173889f; case 23: return -0.19509032368659973f;
    case 24: return 0.0f; case 25: return 0.19509032368659973f; case 26: return 0.38268342614173889f;
    case 27: return 0.55557024478912354f; case 28: return 0.70710676908493042f; case 29: return 0.83146959543228149f;
    case 30: return 0.92387950420379639f; default: return 0.98078525066375732f;
  }
}
PTK_HD constexpr float s32(int m) { return c32(m - 8); }

// (x) * exp(DIR * 2 pi i * m / 32), m compile-time after unrolling; trivial cases cost no multiply
template <int DIR>
PTK_HD cf twiddle32(cf x, int m) {
  m &= 31;
  if (m == 0) return x;
  if (m == 16) return make_float2(-x.x, -x.y);
  if (m == 8) return DIR > 0 ? make_float2(-x.y, x.x) : make_float2(x.y, -x.x);    // * (+-i)
  if (m == 24) return DIR > 0 ? make_float2(x.y, -x.x) : make_float2(-x.y, x.x);
  const float c = c32(m), s = DIR > 0 ? s32(m) : -s32(m);
  return make_float2(fmaf(-x.y, s, x.x * c), fmaf(x.x, s, x.y * c));
}

// in-register DFT of R = 2^k points, natural order in and out.  DIR = -1 forward (exp(-2 pi i ..)), +1 backward.
// Decimation in time, radix 2, constant twiddles; all indices are compile-time after unrolling.  A butterfly with a
// non-trivial twiddle w is written in FMA form: y0 = e + w o (4 FMA), y1 = 2 e - y0 (2 FMA) — 6 instructions instead of
// the 8 of "multiply, then add and subtract".
template <int R, int DIR>
struct Dft {
  static PTK_HD void run(cf* x) {
    cf e[R / 2], o[R / 2];
#pragma unroll
    for (int k = 0; k < R / 2; ++k) { e[k] = x[2 * k]; o[k] = x[2 * k + 1]; }
    Dft<R / 2, DIR>::run(e);
    Dft<R / 2, DIR>::run(o);
#pragma unroll
    for (int k = 0; k < R / 2; ++k) {
      const int m = k * (32 / R);                                 // twiddle exp(DIR 2 pi i m / 32), m < 16
      if (m == 0) {
        x[k] = cadd(e[k], o[k]); x[k + R / 2] = csub(e[k], o[k]);
      } else if (m == 8) {
        const cf t = DIR > 0 ? make_float2(-o[k].y, o[k].x) : make_float2(o[k].y, -o[k].x);   // (+-i) o
        x[k] = cadd(e[k], t); x[k + R / 2] = csub(e[k], t);
      } else {
        const float c = c32(m), sn = DIR > 0 ? s32(m) : -s32(m);
        const cf y0 = make_float2(fmaf(-sn, o[k].y, fmaf(c, o[k].x, e[k].x)), fmaf(sn, o[k].x, fmaf(c, o[k].y, e[k].y)));
        x[k] = y0;
        x[k + R / 2] = make_float2(fmaf(2.0f, e[k].x, -y0.x), fmaf(2.0f, e[k].y, -y0.y));
      }
    }
  }
};
template <int DIR>
struct Dft<1, DIR> { static PTK_HD void run(cf*) {} };

// ---------------------------------------------------------------------------------------------------
template <int N_> struct Geo;
// N = side of the transform one CTA holds in registers; NF = side of the whole field; CL = CTAs per field.
// CL = 4 (NF = 256): a cluster of four CTAs, CTA (a, b) = rank a + 2 b holds the sub-lattice x = 2 x' + a,
// y = 2 y' + b and the four 128 x 128 transforms are combined by one radix-2 x 2 stage over distributed shared
// memory (struct Cross below).
template <> struct Geo<128> {
  static constexpr int N = 128, LOGN = 7, T = 512, N1X = 8, N2X = 16, N1Y = 4, N2Y = 32, LX2 = 4, LY2 = 5, LP2 = 2, LP3 = 1;
  static constexpr int NF = 128, CL = 1;
  static constexpr int PF16 = 10;   // 16-byte prefetch slots per thread beside the exchange buffer (1 CTA / SM)
  static constexpr int HXS = 1;     // the hx propagator tables are staged in shared memory beside the hy tables (2 KB)
};
template <> struct Geo<64> {
  static constexpr int N = 64, LOGN = 6, T = 128, N1X = 8, N2X = 8, N1Y = 4, N2Y = 16, LX2 = 3, LY2 = 4, LP2 = 4, LP3 = 2;
  static constexpr int NF = 64, CL = 1;
  static constexpr int PF16 = 8;    // 4 CTAs / SM: 56 KB each
  static constexpr int HXS = 0;     // no room for them without losing the fourth CTA per SM: hx is read from global memory
};
template <> struct Geo<256> {
  static constexpr int N = 128, LOGN = 7, T = 512, N1X = 8, N2X = 16, N1Y = 4, N2Y = 32, LX2 = 4, LY2 = 5, LP2 = 2, LP3 = 1;
  static constexpr int NF = 256, CL = 4;
  static constexpr int PF16 = 10;
  static constexpr int HXS = 0;     // 4 KB more would exceed the 227 KB of a CTA: hx is read from global memory
};

template <class G>
struct Lay {
  static constexpr int N = G::N, T = G::T;
  struct NoHook { PTK_HD void operator()(int) const {} };
  // The exchange buffer is one region of X1_WARP float2 slots per warp.  X1 (warp-local) lives in the calling
  // warp's region; X2 is laid out so that its "p2" side (warp w holds rows b = w*LP2 .. w*LP2+LP2-1 of every
  // k1y plane) also touches ONLY the calling warp's region: slot(b, k1y, qx) = (b / LP2)*X1_WARP +
  // (b % LP2)*N1Y*X2_ROW + k1y*X2_ROW + qx.  Hence no CTA barrier is needed between an X1 access and a p2-side
  // X2 access of the same warp; only the p3 side (which reads / writes every region) is fenced by CTA barriers.
  static constexpr int X2_ROW = G::N + 8;                 // float2 slots per (b, k1y) row, skewed by 8 (ROW mod 16 = 8)
  static constexpr int X2_WARP = G::LP2 * G::N1Y * X2_ROW;
  static constexpr int X1_WARP = 33 * 32 > X2_WARP ? 33 * 32 : X2_WARP;   // float2 slots per warp region
  static constexpr int XBUF = (T / 32) * X1_WARP;         // float2 slots
  static constexpr int TW = G::N1X * G::N2X + G::N1Y * G::N2Y;   // twiddle table entries (float2)

  // ---- R-layout: thread t, reg r -> (y, x)
  static PTK_HD int r_x(int t, int r) { return (t & (G::N2X - 1)) + G::N2X * (r & (G::N1X - 1)); }
  static PTK_HD int r_y(int t, int r) { return (t >> G::LX2) + G::N2Y * (r / G::N1X); }
  // ---- F-layout: thread t, reg r -> (qy, qx)
  static PTK_HD int f_qx(int t, int) { return t & (N - 1); }
  static PTK_HD int f_qy(int t, int r) { return ((t >> G::LOGN) * G::LP3 + r / G::N2Y) + G::N1Y * (r & (G::N2Y - 1)); }
  // native (coalesced) storage index of (thread, reg) in float2 units — used for every field kept in the
  // workspace, in both layouts.  Registers (2p, 2p+1) of a thread are adjacent, so one thread moves 16 bytes
  // and a warp 512 contiguous bytes per access: as a float4 array the index is p*T + t.
  static PTK_HD int native(int t, int r) { return (((r >> 1) * T + t) << 1) | (r & 1); }
  // position of real-space pixel (y, x) in R-native storage (used by the object-gradient gather)
  static PTK_HD int r_native_of(int y, int x) {
    int a = x & (G::N2X - 1), n1x = x >> G::LX2, b = y & (G::N2Y - 1), n1y = y >> G::LY2;
    return native(a + G::N2X * b, n1y * G::N1X + n1x);
  }
  static PTK_HD int f_native_of(int qy, int qx) {
    int k1y = qy & (G::N1Y - 1), k2y = qy / G::N1Y;
    int c = k1y / G::LP3, ksel = k1y % G::LP3;
    return native(qx + N * c, ksel * G::N2Y + k2y);
  }

  // fill the twiddle table: tw[k1x*N2X + a] = W_N^(a k1x), tw[N1X*N2X + k1y*N2Y + b] = W_N^(b k1y)   (forward sign)
  static PTK_HD void fill_twiddle(cf* tw, int idx) {
    int m;
    if (idx < G::N1X * G::N2X) m = (idx / G::N2X) * (idx % G::N2X);
    else { int i = idx - G::N1X * G::N2X; m = (i / G::N2Y) * (i % G::N2Y); }
    float s, c;
    sincospif(-2.0f * (float)(m % N) / (float)N, &s, &c);
    tw[idx] = make_float2(c, s);
  }

  // ---- phase 1 (forward): R-layout regs -> (k1y, k1x) regs with twiddles.  In two pieces so that a caller can run the row
  // transforms of registers [n1y N1X, (n1y + 1) N1X) as soon as those registers are final (the chain kernels interleave them with
  // the global stores of the pointwise stretch): phase1_fwd = phase1_fwd_row for every n1y, then phase1_fwd_rest.
  static PTK_HD void phase1_fwd_row(cf (&v)[32], int n1y) {
    cf x[G::N1X];
#pragma unroll
    for (int i = 0; i < G::N1X; ++i) x[i] = v[n1y * G::N1X + i];
    Dft<G::N1X, -1>::run(x);
#pragma unroll
    for (int i = 0; i < G::N1X; ++i) v[n1y * G::N1X + i] = x[i];
  }
  static PTK_HD void phase1_fwd(cf (&v)[32], const cf* tw, int t) {
#pragma unroll
    for (int n1y = 0; n1y < G::N1Y; ++n1y) phase1_fwd_row(v, n1y);
    phase1_fwd_rest(v, tw, t);
  }
  static PTK_HD void phase1_fwd_rest(cf (&v)[32], const cf* tw, int t) {
    const int a = t & (G::N2X - 1), b = t >> G::LX2;
#pragma unroll
    for (int k1x = 0; k1x < G::N1X; ++k1x) {
      cf x[G::N1Y];
#pragma unroll
      for (int i = 0; i < G::N1Y; ++i) x[i] = v[i * G::N1X + k1x];
      Dft<G::N1Y, -1>::run(x);
      if (k1x > 0) {
        cf wx = tw[k1x * G::N2X + a];
#pragma unroll
        for (int i = 0; i < G::N1Y; ++i) x[i] = cmul(x[i], wx);
      }
#pragma unroll
      for (int i = 0; i < G::N1Y; ++i) v[i * G::N1X + k1x] = x[i];
    }
#pragma unroll
    for (int k1y = 1; k1y < G::N1Y; ++k1y) {
      cf wy = tw[G::N1X * G::N2X + k1y * G::N2Y + b];
#pragma unroll
      for (int k1x = 0; k1x < G::N1X; ++k1x) v[k1y * G::N1X + k1x] = cmul(v[k1y * G::N1X + k1x], wy);
    }
  }
  // ---- phase 1 (inverse): (k1y, k1x) regs -> R-layout regs.  phase1_inv_h calls hook(step), step = 0 .. N1X + N1Y - 1, between its
  // column and row transforms: the chain kernels issue their asynchronous copies there, a few per step, instead of in one burst
  // before the arithmetic (the copy instructions queue behind one another; spread out, the arithmetic issues meanwhile).
  static PTK_HD void phase1_inv(cf (&v)[32], const cf* tw, int t) { phase1_inv_h(v, tw, t, NoHook()); }
  template <class Hook>
  static PTK_HD void phase1_inv_h(cf (&v)[32], const cf* tw, int t, Hook hook) {
    const int a = t & (G::N2X - 1), b = t >> G::LX2;
#pragma unroll
    for (int k1y = 1; k1y < G::N1Y; ++k1y) {
      cf wy = tw[G::N1X * G::N2X + k1y * G::N2Y + b];
#pragma unroll
      for (int k1x = 0; k1x < G::N1X; ++k1x) v[k1y * G::N1X + k1x] = cmulc(v[k1y * G::N1X + k1x], wy);
    }
#pragma unroll
    for (int k1x = 0; k1x < G::N1X; ++k1x) {
      cf x[G::N1Y];
#pragma unroll
      for (int i = 0; i < G::N1Y; ++i) x[i] = v[i * G::N1X + k1x];
      if (k1x > 0) {
        cf wx = tw[k1x * G::N2X + a];
#pragma unroll
        for (int i = 0; i < G::N1Y; ++i) x[i] = cmulc(x[i], wx);
      }
      Dft<G::N1Y, +1>::run(x);
#pragma unroll
      for (int i = 0; i < G::N1Y; ++i) v[i * G::N1X + k1x] = x[i];
      hook(k1x);
    }
#pragma unroll
    for (int n1y = 0; n1y < G::N1Y; ++n1y) {
      cf x[G::N1X];
#pragma unroll
      for (int i = 0; i < G::N1X; ++i) x[i] = v[n1y * G::N1X + i];
      Dft<G::N1X, +1>::run(x);
#pragma unroll
      for (int i = 0; i < G::N1X; ++i) v[n1y * G::N1X + i] = x[i];
      hook(G::N1X + n1y);
    }
  }
  // ---- phase 2: LP2 lines of N2X points (reg = line*N2X + point)
  template <int DIR>
  static PTK_HD void phase2(cf (&v)[32]) {
#pragma unroll
    for (int l = 0; l < G::LP2; ++l) {
      cf x[G::N2X];
#pragma unroll
      for (int i = 0; i < G::N2X; ++i) x[i] = v[l * G::N2X + i];
      Dft<G::N2X, DIR>::run(x);
#pragma unroll
      for (int i = 0; i < G::N2X; ++i) v[l * G::N2X + i] = x[i];
    }
  }
  // ---- phase 3: LP3 lines of N2Y points
  template <int DIR>
  static PTK_HD void phase3(cf (&v)[32]) {
#pragma unroll
    for (int l = 0; l < G::LP3; ++l) {
      cf x[G::N2Y];
#pragma unroll
      for (int i = 0; i < G::N2Y; ++i) x[i] = v[l * G::N2Y + i];
      Dft<G::N2Y, DIR>::run(x);
#pragma unroll
      for (int i = 0; i < G::N2Y; ++i) v[l * G::N2Y + i] = x[i];
    }
  }

  // ---- exchange X1: warp-local transpose lane <-> reg.  "p1" side: thread t (lane L), reg R = k1y*N1X + k1x.
  // "p2" side: lane L' = R, reg R' = L (= a + N2X*bsel).  slot(L, R) = warp*X1_WARP + R*33 + L.
  static PTK_HD void x1_store_p1(const cf (&v)[32], cf* sm, int t) {
    cf* base = sm + (t >> 5) * X1_WARP + (t & 31);
#pragma unroll
    for (int r = 0; r < 32; ++r) base[r * 33] = v[r];
  }
  static PTK_HD void x1_load_p1(cf (&v)[32], const cf* sm, int t) {
    const cf* base = sm + (t >> 5) * X1_WARP + (t & 31);
#pragma unroll
    for (int r = 0; r < 32; ++r) v[r] = base[r * 33];
  }
  static PTK_HD void x1_store_p2(const cf (&v)[32], cf* sm, int t) {
    cf* base = sm + (t >> 5) * X1_WARP + (t & 31) * 33;
#pragma unroll
    for (int r = 0; r < 32; ++r) base[r] = v[r];
  }
  static PTK_HD void x1_load_p2(cf (&v)[32], const cf* sm, int t) {
    const cf* base = sm + (t >> 5) * X1_WARP + (t & 31) * 33;
#pragma unroll
    for (int r = 0; r < 32; ++r) v[r] = base[r];
  }
  // ---- exchange X2: slot(b, k1y, qx) as above.
  // "p2" side: thread t = warp w, lane (k1y, k1x); reg (bsel, k2x): b = w*LP2 + bsel, qx = k1x + N1X*k2x.
  static PTK_HD int x2_slot(int b, int k1y, int qx) {
    return (b / G::LP2) * X1_WARP + (b % G::LP2) * (G::N1Y * X2_ROW) + k1y * X2_ROW + qx;
  }
  static PTK_HD int x2_base_p2(int t) {
    const int w = t >> 5, k1y = (t & 31) / G::N1X, k1x = t & (G::N1X - 1);
    return w * X1_WARP + k1y * X2_ROW + k1x;
  }
  static PTK_HD int x2_off_p2(int r) { return (r / G::N2X) * (G::N1Y * X2_ROW) + (r & (G::N2X - 1)) * G::N1X; }
  static PTK_HD void x2_store_p2(const cf (&v)[32], cf* sm, int t) {
    cf* base = sm + x2_base_p2(t);
#pragma unroll
    for (int r = 0; r < 32; ++r) base[x2_off_p2(r)] = v[r];
  }
  static PTK_HD void x2_load_p2(cf (&v)[32], const cf* sm, int t) {
    const cf* base = sm + x2_base_p2(t);
#pragma unroll
    for (int r = 0; r < 32; ++r) v[r] = base[x2_off_p2(r)];
  }
  // "p3" side: thread t = (qx, c); reg (ksel, b): k1y = c*LP3 + ksel.
  static PTK_HD int x2_base_p3(int t) { return ((t >> G::LOGN) * G::LP3) * X2_ROW + (t & (N - 1)); }
  static PTK_HD int x2_off_p3(int r) {
    const int ksel = r / G::N2Y, b = r & (G::N2Y - 1);
    return ksel * X2_ROW + (b / G::LP2) * X1_WARP + (b % G::LP2) * (G::N1Y * X2_ROW);
  }
  static PTK_HD void x2_store_p3(const cf (&v)[32], cf* sm, int t) {
    cf* base = sm + x2_base_p3(t);
#pragma unroll
    for (int r = 0; r < 32; ++r) base[x2_off_p3(r)] = v[r];
  }
  static PTK_HD void x2_load_p3(cf (&v)[32], const cf* sm, int t) {
    const cf* base = sm + x2_base_p3(t);
#pragma unroll
    for (int r = 0; r < 32; ++r) v[r] = base[x2_off_p3(r)];
  }
};

// ---------------------------------------------------------------------------------------------------
// Field-level maps (cluster-aware).  For CL = 1 they are Lay's.  For CL = 4 the CTA of rank p = a + 2 b holds
//   real space   : reg r of thread t  <->  pixel (2 r_y(t,r) + b, 2 r_x(t,r) + a)                    ("R-layout")
//   Fourier space: reg r = 8 c + e of thread t, quadrant c = cx + 2 cy, e = 0..7  <->
//                  qx = f_qx(t) + N cx,  qy = f_qy(t, 8 p + e) + N cy                                ("C-layout")
// i.e. after the four sub-lattice transforms, CTA p owns registers [8p, 8p+8) of every thread of all four
// CTAs and combines them into the four frequency quadrants (decimation in time, PAPER-independent textbook
// identity  F[q' + N c] = sum_a (-1)^(a c) W_2N^(a q') F_a[q']  per axis).
// Fields kept in the workspace are stored as [rank][N*N] blocks of Lay::native order in both spaces.
// ---------------------------------------------------------------------------------------------------
template <class G>
struct FL {
  typedef Lay<G> L;
  static constexpr int CL = G::CL, NF = G::NF, NS = G::N, NNS = NS * NS, NNF = NF * NF, NXV = CL == 1 ? 1 : 2;
  static PTK_HD int pix_x(int rank, int t, int r) { return CL == 1 ? L::r_x(t, r) : 2 * L::r_x(t, r) + (rank & 1); }
  static PTK_HD int pix_y(int rank, int t, int r) { return CL == 1 ? L::r_y(t, r) : 2 * L::r_y(t, r) + (rank >> 1); }
  static PTK_HD int fq_xsel(int r) { return CL == 1 ? 0 : (r >> 3) & 1; }       // which of the thread's NXV qx values
  static PTK_HD int fq_x(int rank, int t, int r) { return CL == 1 ? L::f_qx(t, r) : L::f_qx(t, 0) + NS * ((r >> 3) & 1); }
  static PTK_HD int fq_y(int rank, int t, int r) { return CL == 1 ? L::f_qy(t, r) : L::f_qy(t, 8 * rank + (r & 7)) + NS * (r >> 4); }
  // storage index (float2 units, inside one field of NNF elements) of real-space pixel (y, x)
  static PTK_HD int r_native_of(int y, int x) {
    return CL == 1 ? L::r_native_of(y, x) : ((x & 1) + 2 * (y & 1)) * NNS + L::r_native_of(y >> 1, x >> 1);
  }
  // object-pixel offset of register r from the thread's first pixel
  static PTK_HD size_t patch_off(int r, int onx) {
    return (size_t)(CL == 1 ? 1 : 2) * ((size_t)((r / G::N1X) * G::N2Y) * onx + (r & (G::N1X - 1)) * G::N2X);
  }
  // in-place 2 x 2 butterfly over the block index s = r / 8 (self-inverse up to the factor 4)
  static PTK_HD void butterfly(cf (&v)[32]) {
#pragma unroll
    for (int e = 0; e < 8; ++e) {
      const cf s0 = cadd(v[e], v[8 + e]), d0 = csub(v[e], v[8 + e]);
      const cf s1 = cadd(v[16 + e], v[24 + e]), d1 = csub(v[16 + e], v[24 + e]);
      v[e] = cadd(s0, s1); v[8 + e] = cadd(d0, d1); v[16 + e] = csub(s0, s1); v[24 + e] = csub(d0, d1);
    }
  }
  // tw2[m] = exp(-2 pi i m / (2 N)), m < N
  static PTK_HD void fill_tw2(cf* tw2, int m) {
    float s, c;
    sincospif(-(float)m / (float)NS, &s, &c);
    tw2[m] = make_float2(c, s);
  }
  // sub-lattice twiddle W_2N^(a qx' + b qy') on sub-F-layout registers (INV: conjugate)
  template <bool INV>
  static PTK_HD void twiddle(cf (&v)[32], const cf* tw2, int t, int rank) {
    if (CL == 1 || rank == 0) return;
    cf wx = make_float2(1.f, 0.f);
    if (rank & 1) wx = tw2[L::f_qx(t, 0)];
    if (rank >> 1) {
#pragma unroll
      for (int r = 0; r < 32; ++r) { const cf w = cmul(wx, tw2[L::f_qy(t, r)]); v[r] = INV ? cmulc(v[r], w) : cmul(v[r], w); }
    } else {
#pragma unroll
      for (int r = 0; r < 32; ++r) v[r] = INV ? cmulc(v[r], wx) : cmul(v[r], wx);
    }
  }
  // exchange slots in the exchange buffer, float4 units: block src, register pair ep, thread t
  static PTK_HD int xslot(int src, int ep, int t) { return (src * 4 + ep) * G::T + t; }
};

#if defined(__CUDACC__)
// ---- cluster primitives (CL = 4 only)
__device__ __forceinline__ unsigned cluster_ctarank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
// Arrive that only says "this thread has finished READING its CTA's exchange buffer" (write-after-read protection; it publishes
// no data).  barrier.cluster.arrive.release compiles to MEMBAR.ALL.CTA + MEMBAR.ALL.GPU + ERRBAR, and the GPU-scope part waits for
// every global store the thread has in flight (the stash / staging stores of the chain kernels): ncu showed `membar` as 7.7 % of
// the N = 256 kernels' stalls.  Here the CTA-scope fence alone is enough: once it retires, the thread's shared-memory loads have
// returned their values, and a load that has completed cannot be affected by a peer's later remote store, which can only be
// issued after every thread of the cluster has executed this arrive.  (config 4: 7489 -> 7296 ms per step)
__device__ __forceinline__ void cluster_arrive_war() { asm volatile("fence.acq_rel.cta;\n\tbarrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ unsigned mapa_u32(unsigned saddr, unsigned rank) {
  unsigned r; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank)); return r;
}
__device__ __forceinline__ void st_cluster_v4(unsigned addr, cf a, cf b) {
  asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y) : "memory");
}

// Whole transforms for one CTA.  `sm` = exchange buffer (Lay::XBUF float2), `tw` = twiddle table (Lay::TW).
// Buffer protocol (one region of Lay::X1_WARP slots per warp, see Lay): X1 and the p2 side of X2 touch only the
// calling warp's region and are ordered by __syncwarp(); the p3 side of X2 touches every region and is fenced
// by two CTA barriers: one between the stores and the loads of the exchange (a true dependency) and one at the
// end of the forward transform (inside an arithmetic-only stretch, so it costs only the skew between warps),
// after which the whole buffer is free again.  Consequences: fft2_fwd may start whenever the calling warp is done
// with its own region; fft2_inv_head may start after an fft2_fwd or any CTA barrier.  Unnormalised.
template <class G>
__device__ __forceinline__ void fft2_fwd_after_rows(cf (&v)[32], cf* sm, const cf* tw, int t);
template <class G>
__device__ __forceinline__ void fft2_fwd(cf (&v)[32], cf* sm, const cf* tw, int t) {
  typedef Lay<G> L;
#pragma unroll
  for (int n1y = 0; n1y < G::N1Y; ++n1y) L::phase1_fwd_row(v, n1y);
  fft2_fwd_after_rows<G>(v, sm, tw, t);
}
// the forward transform whose phase-1 row transforms the caller has already run (Lay::phase1_fwd_row for every n1y)
template <class G>
__device__ __forceinline__ void fft2_fwd_after_rows(cf (&v)[32], cf* sm, const cf* tw, int t) {
  typedef Lay<G> L;
  L::phase1_fwd_rest(v, tw, t);
  __syncwarp();
  L::x1_store_p1(v, sm, t);
  __syncwarp();
  L::x1_load_p2(v, sm, t);
  L::template phase2<-1>(v);
  __syncwarp();                    // every lane has read its X1 values: the warp's region may be overwritten
  L::x2_store_p2(v, sm, t);
  __syncthreads();
  L::x2_load_p3(v, sm, t);
  if (G::CL > 1) cluster_arrive_war();  // this thread no longer reads the exchange buffer: peers may overwrite it (Cross)
  L::template phase3<-1>(v);
  __syncthreads();                 // all p3-side reads are long done: the buffer is free for the next transform.
                                   // Placed after the arithmetic, not after the loads: a barrier behind a burst of
                                   // LDS releases only when the LAST warp got its loads into the queue (~1k cycles)
}
// The inverse in two pieces: after the head, the calling warp's own region (Lay::X1_WARP float2 slots at
// sm + warp*X1_WARP) is free until that warp's next fft2_fwd / fft2_inv_head — the chain kernels land their
// late cp.async prefetches there while phase 1 runs.
template <class G>
__device__ __forceinline__ void fft2_inv_head(cf (&v)[32], cf* sm, int t) {
  typedef Lay<G> L;
  L::template phase3<+1>(v);
  if (G::CL > 1) __syncthreads();  // Cross::inv: other warps may still be reading what peers sent into this buffer
  L::x2_store_p3(v, sm, t);
  __syncthreads();
  L::x2_load_p2(v, sm, t);
  L::template phase2<+1>(v);
  __syncwarp();                    // own-region X2 reads done before the warp-local X1 exchange overwrites them
  L::x1_store_p2(v, sm, t);
  __syncwarp();
  L::x1_load_p1(v, sm, t);
  __syncwarp();                    // every lane has read its part: the warp's region is free
}
template <class G>
__device__ __forceinline__ void fft2_inv(cf (&v)[32], cf* sm, const cf* tw, int t) {
  fft2_inv_head<G>(v, sm, t);
  Lay<G>::phase1_inv(v, tw, t);
}

// ---------------------------------------------------------------------------------------------------
// Cross-CTA radix-2 x 2 stage of the CL = 4 field transform, over distributed shared memory.
// Every CTA sends registers [8 d, 8 d + 8) of each thread to CTA d (its own block included, through the same
// path) with 16-byte remote stores into the destination's exchange buffer, slot FL::xslot(source, pair, t):
// a warp writes 512 contiguous bytes.  One hardware cluster barrier phase protects the buffer before the
// stores (write-after-read: the matching arrive is issued as soon as a thread has finished reading the
// buffer) and one makes them visible.  Protocol invariant: whenever the registers are in Fourier space
// (C-layout), exactly one cluster arrive of this thread is pending.
// ---------------------------------------------------------------------------------------------------
template <class G>
struct Cross {
  typedef FL<G> F;
  static __device__ __forceinline__ void send(const cf (&v)[32], cf* sm, int t, unsigned rank) {
    const unsigned base = (unsigned)__cvta_generic_to_shared((float4*)sm + F::xslot((int)rank, 0, t));
#pragma unroll
    for (int d = 0; d < 4; ++d) {
      const unsigned ra = mapa_u32(base, (unsigned)d);
#pragma unroll
      for (int ep = 0; ep < 4; ++ep) st_cluster_v4(ra + (unsigned)(ep * G::T * 16), v[8 * d + 2 * ep], v[8 * d + 2 * ep + 1]);
    }
  }
  static __device__ __forceinline__ void recv(cf (&v)[32], const cf* sm, int t) {
    const float4* b = (const float4*)sm;
#pragma unroll
    for (int s = 0; s < 4; ++s)
#pragma unroll
      for (int ep = 0; ep < 4; ++ep) {
        const float4 q = b[F::xslot(s, ep, t)];
        v[8 * s + 2 * ep] = make_float2(q.x, q.y);
        v[8 * s + 2 * ep + 1] = make_float2(q.z, q.w);
      }
  }
  // sub-F-layout (after fft2_fwd, whose last exchange-buffer read issued the pending arrive) -> C-layout
  static __device__ __forceinline__ void fwd(cf (&v)[32], cf* sm, const cf* tw2, int t, unsigned rank) {
    F::template twiddle<false>(v, tw2, t, (int)rank);
    cluster_wait();
    send(v, sm, t, rank);
    cluster_arrive();
    cluster_wait();
    recv(v, sm, t);
    cluster_arrive_war();
    F::butterfly(v);
  }
  // C-layout -> sub-F-layout (ready for fft2_inv_head); consumes the pending arrive
  static __device__ __forceinline__ void inv(cf (&v)[32], cf* sm, const cf* tw2, int t, unsigned rank) {
    F::butterfly(v);
    cluster_wait();
    send(v, sm, t, rank);
    cluster_arrive();
    cluster_wait();
    recv(v, sm, t);
    F::template twiddle<true>(v, tw2, t, (int)rank);
  }
};

// Field-level transforms of one CTA (of a CL-cluster): R-layout <-> Fourier layout (F-layout / C-layout)
template <class G>
struct Fft {
  static __device__ __forceinline__ unsigned rank() { return G::CL > 1 ? cluster_ctarank() : 0u; }
  static __device__ __forceinline__ void begin_fourier() { if (G::CL > 1) cluster_arrive_war(); }   // registers (re)start in Fourier space
  static __device__ __forceinline__ void end_fourier() { if (G::CL > 1) cluster_wait(); }       // kernel ends in Fourier space
  static __device__ __forceinline__ void fwd(cf (&v)[32], cf* sm, const cf* tw, const cf* tw2, int t, unsigned rk) {
    fft2_fwd<G>(v, sm, tw, t);
    if (G::CL > 1) Cross<G>::fwd(v, sm, tw2, t, rk);
  }
  static __device__ __forceinline__ void fwd_after_rows(cf (&v)[32], cf* sm, const cf* tw, const cf* tw2, int t, unsigned rk) {
    fft2_fwd_after_rows<G>(v, sm, tw, t);
    if (G::CL > 1) Cross<G>::fwd(v, sm, tw2, t, rk);
  }
  static __device__ __forceinline__ void inv_head(cf (&v)[32], cf* sm, const cf* tw2, int t, unsigned rk) {
    if (G::CL > 1) Cross<G>::inv(v, sm, tw2, t, rk);
    fft2_inv_head<G>(v, sm, t);
  }
  static __device__ __forceinline__ void inv(cf (&v)[32], cf* sm, const cf* tw, const cf* tw2, int t, unsigned rk) {
    inv_head(v, sm, tw2, t, rk);
    Lay<G>::phase1_inv(v, tw, t);
  }
};
#endif

}  // namespace ptk
