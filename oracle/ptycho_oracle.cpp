// ptycho_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, double-precision CPU restatement of one forward+adjoint iteration of the
// mixed-state multislice ptychography model of arxiv 2505.14372 ("phaser"), written from the
// paper and from the readings R1..R29 listed in DESIGN.md §3.  It shares no code,
// header, table or constant generator with the CUDA path in paper_2505_14372_b200/csrc and
// neither side includes the other.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference leg may load this library.
//
// Everything is the plain definition: naive O(N^2) 1-D DFT (row-column for 2-D) and a simple
// recursive radix-2 FFT, std::complex<double>, no blocking, no fusion.  OpenMP only splits the
// loop over probe positions ("operates on a group of probe positions in parallel").
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): brute-force DFT, Parseval, identity
// propagator at dz=0, propagator composition, integer tilt shift, vacuum-object invariant, SPOA
// special case, phase-ramp object, loss closed forms, dot-product adjoint tests, central finite
// differences of the whole loss, zero gradient at the truth, torch.fft+autograd (complex128)
// cross-check, LSQML line-search optimum, and for the later additions (ePIE, per-position-alpha LSQML update, probe
// preconditioner, regularisers, constraints, Adam) the closed forms, finite differences and numpy restatements named
// beside each function.  "Absolute values vs the paper": parity unpinned —
// the paper prints no numeric example.
//
// Notation follows PAPER.md §III: probe modes P_k, object slices O_i with gaps dz_i, positions
// X_j, exit waves Psi_{i,k}, measured I_exp.  F is the unnormalised forward DFT
// (F a)[q] = sum_r a[r] exp(-2 pi i (qy y + qx x)/N), Finv = F^H / N^2.

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;
static const double PI = 3.14159265358979323846264338327950288;

extern "C" {

// ------------------------------------------------------------------------------------------
// problem description (mirrors the paper's problem statement)
// ------------------------------------------------------------------------------------------
struct orc_problem {
  int32_t n;                 // N, probe / pattern side
  int32_t n_modes;           // M incoherent probe modes
  int32_t n_slices;          // S object slices
  int32_t obj_ny, obj_nx;    // object slice size (px)
  int32_t n_pos_total;       // rows of positions / intensity
  int32_t n_batch;           // J positions in this group
  float pixel_size;          // Angstrom / px (float32: the same value the GPU receives)
  float wavelength;          // Angstrom
  const float* slice_thickness;  // S entries, last unused (reading R10)
  float tilt_x_mrad, tilt_y_mrad;  // propagator tilt (reading R8)
  float bandlimit;           // fraction of Nyquist, <=0: off (reading R9)
  int32_t loss;              // 0 amplitude, 1 Poisson, 2 Gaussian
  float loss_c;              // c of the variance-stabilising transform; Gaussian: sigma
  float eps;                 // epsilon offset (readings R11..R13)
  float lsqml_delta_o;       // delta_O of PAPER.md:219
  float lsqml_delta_p;       // probe analogue (reading R19)
  int32_t shift_mode;        // 0: Fourier shift of the probe (reading R1, default); 1: bilinear sampling of the object
  float lsqml_chi_scale;     // LSQML wavefront update chi = -lsqml_chi_scale * gPhi: 1 = steepest descent (reading R20);
                             // 2 = the modulus-constraint update of PAPER.md:173, (ae/(eps+a) - 1) psi~ = -2 w psi~ (reading R31,
                             // amplitude loss only)
};

// ------------------------------------------------------------------------------------------
// DFT / FFT
// ------------------------------------------------------------------------------------------
// naive 1-D DFT, sign=-1 forward, +1 backward (unnormalised). stride in elements.
static void dft1_naive(int n, const cd* in, int sin, cd* out, int sout, int sign) {
  for (int k = 0; k < n; ++k) {
    cd acc = 0.0;
    for (int r = 0; r < n; ++r) {
      // reduce k*r mod n before forming the angle so the argument stays accurate
      long kr = ((long)k * (long)r) % n;
      double ang = sign * 2.0 * PI * (double)kr / (double)n;
      acc += in[(long)r * sin] * cd(std::cos(ang), std::sin(ang));
    }
    out[(long)k * sout] = acc;
  }
}

// simple recursive radix-2 decimation-in-time FFT, n power of two, unnormalised
static void fft1_rec(int n, const cd* in, int sin, cd* out, int sign) {
  if (n == 1) { out[0] = in[0]; return; }
  int h = n / 2;
  std::vector<cd> ev(h), od(h);
  fft1_rec(h, in, sin * 2, ev.data(), sign);
  fft1_rec(h, in + sin, sin * 2, od.data(), sign);
  for (int k = 0; k < h; ++k) {
    double ang = sign * 2.0 * PI * (double)k / (double)n;
    cd t = cd(std::cos(ang), std::sin(ang)) * od[k];
    out[k] = ev[k] + t;
    out[k + h] = ev[k] - t;
  }
}

static bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// 2-D transform of an n x n row-major field, in place. naive!=0 uses the O(n^2) 1-D DFT.
static void xform2(int n, cd* a, int sign, int naive) {
  std::vector<cd> line(n), res(n);
  for (int y = 0; y < n; ++y) {           // rows (x direction)
    for (int x = 0; x < n; ++x) line[x] = a[(long)y * n + x];
    if (naive || !is_pow2(n)) dft1_naive(n, line.data(), 1, res.data(), 1, sign);
    else fft1_rec(n, line.data(), 1, res.data(), sign);
    for (int x = 0; x < n; ++x) a[(long)y * n + x] = res[x];
  }
  for (int x = 0; x < n; ++x) {           // columns (y direction)
    for (int y = 0; y < n; ++y) line[y] = a[(long)y * n + x];
    if (naive || !is_pow2(n)) dft1_naive(n, line.data(), 1, res.data(), 1, sign);
    else fft1_rec(n, line.data(), 1, res.data(), sign);
    for (int y = 0; y < n; ++y) a[(long)y * n + x] = res[y];
  }
}
static void F2(int n, cd* a) { xform2(n, a, -1, 0); }
static void Finv2(int n, cd* a) {
  xform2(n, a, +1, 0);
  double s = 1.0 / ((double)n * (double)n);
  for (long i = 0; i < (long)n * n; ++i) a[i] *= s;
}

// exported for the pins: out = F(in) (sign=-1) or F^H(in) (sign=+1), unnormalised
void orc_dft2_naive(int32_t n, const double* in, double* out, int32_t sign) {
  std::vector<cd> a((long)n * n);
  for (long i = 0; i < (long)n * n; ++i) a[i] = cd(in[2 * i], in[2 * i + 1]);
  xform2(n, a.data(), sign, 1);
  for (long i = 0; i < (long)n * n; ++i) { out[2 * i] = a[i].real(); out[2 * i + 1] = a[i].imag(); }
}
// direct O(N^4) double sum, no row-column split (for 8x8 brute force)
void orc_dft2_bruteforce(int32_t n, const double* in, double* out, int32_t sign) {
  for (int qy = 0; qy < n; ++qy)
    for (int qx = 0; qx < n; ++qx) {
      cd acc = 0.0;
      for (int y = 0; y < n; ++y)
        for (int x = 0; x < n; ++x) {
          double ang = sign * 2.0 * PI * ((double)(qy * y) + (double)(qx * x)) / (double)n;
          acc += cd(in[2 * ((long)y * n + x)], in[2 * ((long)y * n + x) + 1]) * cd(std::cos(ang), std::sin(ang));
        }
      out[2 * ((long)qy * n + qx)] = acc.real();
      out[2 * ((long)qy * n + qx) + 1] = acc.imag();
    }
}
void orc_fft2(int32_t n, const double* in, double* out, int32_t sign) {
  std::vector<cd> a((long)n * n);
  for (long i = 0; i < (long)n * n; ++i) a[i] = cd(in[2 * i], in[2 * i + 1]);
  xform2(n, a.data(), sign, 0);
  for (long i = 0; i < (long)n * n; ++i) { out[2 * i] = a[i].real(); out[2 * i + 1] = a[i].imag(); }
}

// signed frequency in cycles / px: f(n) = n/N for n < N/2, (n-N)/N otherwise (Nyquist at -1/2)
static double freq(int n, int N) { return (n < N / 2) ? (double)n / N : (double)(n - N) / N; }

// ------------------------------------------------------------------------------------------
// O1: position split, reading R2 — done in float32, the same arithmetic as the GPU, so a
// rounding flip at a half pixel cannot break parity; promoted to double afterwards.
// ------------------------------------------------------------------------------------------
void orc_position_split(float X, float px, int32_t N, int32_t* r0, float* delta) {
  volatile float p = X / px;
  volatile float c = p - (float)(N / 2);
  volatile float ch = c + 0.5f;
  float fl = std::floor(ch);
  volatile float d = c - fl;
  *r0 = (int32_t)fl;
  *delta = d;
}

// O1 (bilinear mode, reading R1 secondary): c = X/px - N/2, i0 = floor(c), f = c - i0 in [0,1), float32 as above
void orc_position_split_floor(float X, float px, int32_t N, int32_t* i0, float* frac) {
  volatile float p = X / px;
  volatile float c = p - (float)(N / 2);
  float fl = std::floor(c);
  volatile float d = c - fl;
  *i0 = (int32_t)fl;
  *frac = d;
}

// O3 (bilinear mode): the four taps of window pixel (y, x): object pixels (i0 + r + d), d in {0,1}^2, with weights
// w_d = (d_y ? f_y : 1 - f_y)(d_x ? f_x : 1 - f_x)   ("sampled")
static inline double bil_w(int d, double f) { return d ? f : 1.0 - f; }

// O1: sub-pixel shift ramp R[q] = exp(-2 pi i (f(qy) dy + f(qx) dx))  (PAPER.md:115 P_k(r - X_j))
static void shift_ramp(int N, double dy, double dx, cd* R) {
  for (int qy = 0; qy < N; ++qy)
    for (int qx = 0; qx < N; ++qx) {
      double ang = -2.0 * PI * (freq(qy, N) * dy + freq(qx, N) * dx);
      R[(long)qy * N + qx] = cd(std::cos(ang), std::sin(ang));
    }
}

// O4: Fresnel propagator with tilt and band limit (readings R7,R8,R9)
// H[q] = B[q] exp(-i pi lambda dz (kx^2+ky^2)) exp(+2 pi i dz (kx tan tx + ky tan ty))
static void propagator(int N, double px, double lambda, double dz, double tx_mrad, double ty_mrad,
                       double bandlimit, cd* H) {
  double tx = std::tan(tx_mrad * 1e-3), ty = std::tan(ty_mrad * 1e-3);
  for (int qy = 0; qy < N; ++qy)
    for (int qx = 0; qx < N; ++qx) {
      double fy = freq(qy, N), fx = freq(qx, N);
      double ky = fy / px, kx = fx / px;   // cycles / Angstrom
      double ang = -PI * lambda * dz * (kx * kx + ky * ky) + 2.0 * PI * dz * (kx * tx + ky * ty);
      double B = 1.0;
      if (bandlimit > 0.0) {
        // sharp inclusive circular mask at bandlimit x Nyquist; compared on integer frequency
        // indices (exact) against (0.5*bandlimit*N)^2
        int iy = (qy < N / 2) ? qy : qy - N, ix = (qx < N / 2) ? qx : qx - N;
        double lim = 0.5 * bandlimit * N;
        B = ((double)(iy * iy + ix * ix) <= lim * lim) ? 1.0 : 0.0;
      }
      H[(long)qy * N + qx] = B * cd(std::cos(ang), std::sin(ang));
    }
}
void orc_propagator(int32_t N, double px, double lambda, double dz, double tx_mrad, double ty_mrad,
                    double bandlimit, double* H_out) {
  std::vector<cd> H((long)N * N);
  propagator(N, px, lambda, dz, tx_mrad, ty_mrad, bandlimit, H.data());
  for (long i = 0; i < (long)N * N; ++i) { H_out[2 * i] = H[i].real(); H_out[2 * i + 1] = H[i].imag(); }
}

// ------------------------------------------------------------------------------------------
// The linear pieces of the model.  forward_pos / adjoint_pos / orc_gradient below call exactly these
// helpers, and the exported orc_shift / orc_propagate / orc_gather / orc_scatter_add wrappers call them
// too, so the dot-product and coverage-map pins (tests/test_oracle_pins.py) run the model's own code.
// ------------------------------------------------------------------------------------------
// a[q] *= R[q]  (adjoint: conj(R[q]))                    — Fourier side of O2 / O9
static void mul_ramp(long NN, cd* a, const cd* R, bool adjoint) {
  for (long q = 0; q < NN; ++q) a[q] *= adjoint ? std::conj(R[q]) : R[q];
}
// a <- Finv(H .* F(a))  (adjoint: Finv(conj(H) .* F(a)))  — O3 / O8
static void propagate_field(int N, cd* a, const cd* H, bool adjoint) {
  F2(N, a);
  for (long q = 0; q < (long)N * N; ++q) a[q] *= adjoint ? std::conj(H[q]) : H[q];
  Finv2(N, a);
}
// patch[r] = slice[r0 + r]   (O3); slice = one object slice [ony][onx]
static void gather_window(int N, int onx, const cd* slice, int r0y, int r0x, cd* patch) {
  for (int y = 0; y < N; ++y)
    for (int x = 0; x < N; ++x) patch[(long)y * N + x] = slice[(long)(r0y + y) * onx + (r0x + x)];
}
// slice[r0 + r] += patch[r]  (O8 last line)
static void scatter_add_window(int N, int onx, cd* slice, int r0y, int r0x, const cd* patch) {
  for (int y = 0; y < N; ++y)
    for (int x = 0; x < N; ++x) slice[(long)(r0y + y) * onx + (r0x + x)] += patch[(long)y * N + x];
}
// bilinear variants (reading R1 secondary): patch[r] = sum_d w_d slice[i0 + r + d] and its adjoint
static void gather_window_bilinear(int N, int onx, const cd* slice, int i0y, int i0x, double fy, double fx, cd* patch) {
  for (int y = 0; y < N; ++y)
    for (int x = 0; x < N; ++x) {
      cd acc = 0.0;
      for (int dy = 0; dy < 2; ++dy)
        for (int dx = 0; dx < 2; ++dx)
          acc += bil_w(dy, fy) * bil_w(dx, fx) * slice[(long)(i0y + y + dy) * onx + (i0x + x + dx)];
      patch[(long)y * N + x] = acc;
    }
}
static void scatter_add_window_bilinear(int N, int onx, cd* slice, int i0y, int i0x, double fy, double fx, const cd* patch) {
  for (int y = 0; y < N; ++y)
    for (int x = 0; x < N; ++x)
      for (int dy = 0; dy < 2; ++dy)
        for (int dx = 0; dx < 2; ++dx)
          slice[(long)(i0y + y + dy) * onx + (i0x + x + dx)] += bil_w(dy, fy) * bil_w(dx, fx) * patch[(long)y * N + x];
}

static std::vector<cd> to_cd(const double* in, long n) {
  std::vector<cd> a(n);
  for (long i = 0; i < n; ++i) a[i] = cd(in[2 * i], in[2 * i + 1]);
  return a;
}
static void from_cd(const std::vector<cd>& a, double* out) {
  for (size_t i = 0; i < a.size(); ++i) { out[2 * i] = a[i].real(); out[2 * i + 1] = a[i].imag(); }
}
// exported for the pins ---------------------------------------------------------------------
// out = Finv(R(dy,dx) .* F(in))        (O2 with in = P_k; adjoint: conj(R))
void orc_shift(int32_t N, const double* in, double dy, double dx, double* out, int32_t adjoint) {
  std::vector<cd> a = to_cd(in, (long)N * N), R((long)N * N);
  shift_ramp(N, dy, dx, R.data());
  F2(N, a.data());
  mul_ramp((long)N * N, a.data(), R.data(), adjoint != 0);
  Finv2(N, a.data());
  from_cd(a, out);
}
// out = Finv(H .* F(in)), or with adjoint: Finv(conj(H) .* F(in))   (O3 / O8)
void orc_propagate(int32_t N, const double* in, double px, double lambda, double dz, double tx_mrad,
                   double ty_mrad, double bandlimit, double* out, int32_t adjoint) {
  std::vector<cd> a = to_cd(in, (long)N * N), H((long)N * N);
  propagator(N, px, lambda, dz, tx_mrad, ty_mrad, bandlimit, H.data());
  propagate_field(N, a.data(), H.data(), adjoint != 0);
  from_cd(a, out);
}
// patch[r] = obj[r0 + r]   (O3)
void orc_gather(int32_t N, int32_t ony, int32_t onx, const double* obj, int32_t r0y, int32_t r0x, double* patch) {
  std::vector<cd> o = to_cd(obj, (long)ony * onx), pt((long)N * N);
  gather_window(N, onx, o.data(), r0y, r0x, pt.data());
  from_cd(pt, patch);
}
// obj[r0 + r] += patch[r]  (O8 last line)
void orc_scatter_add(int32_t N, int32_t ony, int32_t onx, double* obj, int32_t r0y, int32_t r0x, const double* patch) {
  std::vector<cd> o = to_cd(obj, (long)ony * onx), pt = to_cd(patch, (long)N * N);
  scatter_add_window(N, onx, o.data(), r0y, r0x, pt.data());
  from_cd(o, obj);
}

// patch[r] = sum_d w_d obj[i0 + r + d]; with adjoint != 0: obj[i0 + r + d] += w_d patch[r]   (exported for the pins)
void orc_bilinear(int32_t N, int32_t ony, int32_t onx, double* obj, int32_t i0y, int32_t i0x, double fy, double fx,
                  double* patch, int32_t adjoint) {
  std::vector<cd> o = to_cd(obj, (long)ony * onx);
  if (adjoint) {
    std::vector<cd> pt = to_cd(patch, (long)N * N);
    scatter_add_window_bilinear(N, onx, o.data(), i0y, i0x, fy, fx, pt.data());
    from_cd(o, obj);
  } else {
    std::vector<cd> pt((long)N * N);
    gather_window_bilinear(N, onx, o.data(), i0y, i0x, fy, fx, pt.data());
    from_cd(pt, patch);
  }
}

// O6: per-pixel loss l(I, Iexp) and detector weight w = dl/dI
// Poisson (PAPER.md:151 Stirling form, epsilon inside both logarithms — reading R11; w = PAPER.md:165)
// Amplitude/Anscombe (PAPER.md:157 as printed; w = its derivative regularised as PAPER.md:167 — reading R12)
// Gaussian: l = (I - Iexp)^2 / (2 sigma^2), normalisation constant dropped as the paper says;
// sigma is passed in the c slot; w = (I - Iexp) / sigma^2
void orc_loss_pixel(int32_t kind, double I, double Iexp, double c, double eps, double* l, double* w) {
  if (kind == 2) {
    *l = (I - Iexp) * (I - Iexp) / (2.0 * c * c);
    *w = (I - Iexp) / (c * c);
  } else if (kind == 1) {
    *l = I - Iexp * (std::log(I + eps) - std::log(Iexp + eps) + 1.0);
    *w = 1.0 - Iexp / (I + eps);
  } else {
    double a = std::sqrt(I + c), ae = std::sqrt(Iexp + c);
    *l = 0.5 * (a - ae) * (a - ae);
    *w = 0.5 * (1.0 - ae / (a + eps));
  }
}

}  // extern "C" (helpers below are C++)

// ------------------------------------------------------------------------------------------
// one position: forward (O1..O6) and, optionally, adjoint (O7..O10)
// ------------------------------------------------------------------------------------------
struct PosWork {
  int N, M, S;
  std::vector<cd> R;                 // shift ramp
  std::vector<std::vector<cd>> Psi;  // [i*M+k] entering wave of slice i, mode k
  std::vector<std::vector<cd>> T;    // [i] object patch
  std::vector<std::vector<cd>> psit; // [k] far field / N
  std::vector<std::vector<cd>> gPhi; // [i*M+k] gradient wrt the exit wave of slice i (only kept when asked)
  std::vector<double> I;
  int r0y, r0x; double dy, dx;
};

struct Model {
  orc_problem p;
  int N, M, S;
  long NN;
  std::vector<std::vector<cd>> Pt;   // F(P_k)           (O0)
  std::vector<std::vector<cd>> H;    // H_i, i<S-1       (O4)
  std::vector<cd> obj;               // [S][ony][onx]
  const float* positions; const float* intensity; const int32_t* batch_idx;
};

static void model_init(Model& m, const orc_problem* p, const float* object, const float* probe,
                       const float* positions, const float* intensity, const int32_t* batch_idx) {
  m.p = *p; m.N = p->n; m.M = p->n_modes; m.S = p->n_slices; m.NN = (long)p->n * p->n;
  m.positions = positions; m.intensity = intensity; m.batch_idx = batch_idx;
  long on = (long)p->n_slices * p->obj_ny * p->obj_nx;
  m.obj.resize(on);
  for (long i = 0; i < on; ++i) m.obj[i] = cd(object[2 * i], object[2 * i + 1]);
  m.Pt.assign(m.M, std::vector<cd>(m.NN));
  for (int k = 0; k < m.M; ++k) {
    for (long i = 0; i < m.NN; ++i) m.Pt[k][i] = cd(probe[2 * (k * m.NN + i)], probe[2 * (k * m.NN + i) + 1]);
    F2(m.N, m.Pt[k].data());                                                    // O0
  }
  m.H.assign(m.S > 1 ? m.S - 1 : 0, std::vector<cd>(m.NN));
  for (int i = 0; i + 1 < m.S; ++i)
    propagator(m.N, (double)p->pixel_size, (double)p->wavelength, (double)p->slice_thickness[i],
               (double)p->tilt_x_mrad, (double)p->tilt_y_mrad, (double)p->bandlimit, m.H[i].data());
}

// returns 0, or -1 if the window leaves the object (reading R4)
static int forward_pos(const Model& m, int jrow, PosWork& w) {
  const int N = m.N, M = m.M, S = m.S; const long NN = m.NN;
  const orc_problem& p = m.p;
  w.N = N; w.M = M; w.S = S;
  float dyf, dxf; int32_t r0y, r0x;
  const bool bil = p.shift_mode == 1;
  if (!bil) {
    orc_position_split(m.positions[2 * jrow + 0], p.pixel_size, N, &r0y, &dyf);   // O1
    orc_position_split(m.positions[2 * jrow + 1], p.pixel_size, N, &r0x, &dxf);
    if (r0y < 0 || r0x < 0 || r0y + N > p.obj_ny || r0x + N > p.obj_nx) return -1;
  } else {                                                                        // taps i0 .. i0 + N inclusive
    orc_position_split_floor(m.positions[2 * jrow + 0], p.pixel_size, N, &r0y, &dyf);
    orc_position_split_floor(m.positions[2 * jrow + 1], p.pixel_size, N, &r0x, &dxf);
    if (r0y < 0 || r0x < 0 || r0y + N + 1 > p.obj_ny || r0x + N + 1 > p.obj_nx) return -1;
  }
  w.r0y = r0y; w.r0x = r0x; w.dy = (double)dyf; w.dx = (double)dxf;
  w.R.resize(NN); shift_ramp(N, bil ? 0.0 : w.dy, bil ? 0.0 : w.dx, w.R.data());    // bilinear mode: probe unshifted, R = 1
  w.Psi.assign((long)S * M, std::vector<cd>()); w.T.assign(S, std::vector<cd>(NN));
  w.psit.assign(M, std::vector<cd>(NN)); w.I.assign(NN, 0.0);
  const long os = (long)p.obj_ny * p.obj_nx;
  for (int i = 0; i < S; ++i) {                                                  // O3: T_i[r] = O_i[r0 + r]
    if (!bil) gather_window(N, p.obj_nx, m.obj.data() + i * os, r0y, r0x, w.T[i].data());
    else gather_window_bilinear(N, p.obj_nx, m.obj.data() + i * os, r0y, r0x, w.dy, w.dx, w.T[i].data());
  }
  for (int k = 0; k < M; ++k) {
    std::vector<cd> cur = m.Pt[k];
    mul_ramp(NN, cur.data(), w.R.data(), false);                                 // O2: Psi_0 = Finv(R .* P~_k)
    Finv2(N, cur.data());
    for (int i = 0; i < S; ++i) {
      w.Psi[(long)i * M + k] = cur;                                              // entering wave Psi_{i,k}
      for (long r = 0; r < NN; ++r) cur[r] *= w.T[i][r];                         // Phi_{i,k} = Psi .* T
      if (i < S - 1) propagate_field(N, cur.data(), m.H[i].data(), false);       // O3 propagate (reading R10: none after the last slice)
    }
    F2(N, cur.data());                                                           // O5 far field, orthonormal (reading R5)
    for (long q = 0; q < NN; ++q) { cur[q] /= (double)N; w.I[q] += std::norm(cur[q]); }
    w.psit[k] = cur;
  }
  return 0;
}

// adjoint O7..O10 for one position. gT[i] (N x N) is overwritten; gPt_acc[k] += conj(R) .* G~_k;
// gdelta[2] = dL/d(delta_y, delta_x).  If keep_gphi, w.gPhi[i*M+k] keeps gPhi_{i,k} (for O14).
static void adjoint_pos(const Model& m, int jrow, PosWork& w, double* loss_j,
                        std::vector<std::vector<cd>>& gT, std::vector<std::vector<cd>>* gPt_acc,
                        double* gdelta, bool keep_gphi) {
  const int N = m.N, M = m.M, S = m.S; const long NN = m.NN; const orc_problem& p = m.p;
  std::vector<double> wdet(NN);
  double L = 0.0;
  const float* Iexp = m.intensity + (long)jrow * NN;
  for (long q = 0; q < NN; ++q) {                                                // O6
    double l, ww; orc_loss_pixel(p.loss, w.I[q], (double)Iexp[q], (double)p.loss_c, (double)p.eps, &l, &ww);
    L += l; wdet[q] = ww;
  }
  *loss_j = L;
  gT.assign(S, std::vector<cd>(NN, cd(0.0)));
  if (keep_gphi) w.gPhi.assign((long)S * M, std::vector<cd>());
  gdelta[0] = gdelta[1] = 0.0;
  for (int k = 0; k < M; ++k) {
    std::vector<cd> g(NN);
    for (long q = 0; q < NN; ++q) g[q] = wdet[q] * w.psit[k][q];                 // O7: g~ = w .* psi~
    Finv2(N, g.data());
    for (long r = 0; r < NN; ++r) g[r] *= (double)N;                             //     gPhi_{S-1} = N Finv(g~)
    for (int i = S - 1; i >= 0; --i) {                                           // O8
      if (keep_gphi) w.gPhi[(long)i * M + k] = g;
      const std::vector<cd>& Psi = w.Psi[(long)i * M + k];
      for (long r = 0; r < NN; ++r) gT[i][r] += std::conj(Psi[r]) * g[r];        // gT_i += conj(Psi) .* gPhi
      for (long r = 0; r < NN; ++r) g[r] = std::conj(w.T[i][r]) * g[r];          // gPsi = conj(T) .* gPhi
      if (i > 0) propagate_field(N, g.data(), m.H[i - 1].data(), true);          // gPhi_{i-1} = Finv(conj(H_{i-1}) .* F(gPsi_i))
    }
    F2(N, g.data());                                                             // O9: G~ = F(gPsi_0)
    if (gPt_acc) {
      std::vector<cd> c = g;
      mul_ramp(NN, c.data(), w.R.data(), true);                                  //     gP~_k += conj(R) .* G~
      for (long q = 0; q < NN; ++q) (*gPt_acc)[k][q] += c[q];
    }
    for (int a = 0; a < 2 && p.shift_mode != 1; ++a) {                           // O10 (Fourier-shift mode)
      cd acc = 0.0;
      for (int qy = 0; qy < N; ++qy)
        for (int qx = 0; qx < N; ++qx) {
          long q = (long)qy * N + qx;
          double fa = (a == 0) ? freq(qy, N) : freq(qx, N);
          acc += std::conj(g[q]) * cd(0.0, -2.0 * PI * fa) * w.R[q] * m.Pt[k][q];
        }
      gdelta[a] += 2.0 * acc.real() / ((double)N * N);
    }
  }
  if (p.shift_mode == 1) {
    // O10 (bilinear mode): the position enters through the weights only, integer corner held fixed (reading R17):
    // dL/df_a = 2 Re sum_i sum_r conj(gT_i[r]) dT_i[r]/df_a,
    // dT/df_y = sum_dx w_dx (O[y+1, x+dx] - O[y, x+dx]),  dT/df_x = sum_dy w_dy (O[y+dy, x+1] - O[y+dy, x])
    for (int i = 0; i < S; ++i)
      for (int y = 0; y < N; ++y)
        for (int x = 0; x < N; ++x) {
          auto O = [&](int dy, int dx) { return m.obj[((long)i * p.obj_ny + (w.r0y + y + dy)) * p.obj_nx + (w.r0x + x + dx)]; };
          cd dTy = bil_w(0, w.dx) * (O(1, 0) - O(0, 0)) + bil_w(1, w.dx) * (O(1, 1) - O(0, 1));
          cd dTx = bil_w(0, w.dy) * (O(0, 1) - O(0, 0)) + bil_w(1, w.dy) * (O(1, 1) - O(1, 0));
          cd g = gT[i][(long)y * N + x];
          gdelta[0] += 2.0 * (std::conj(g) * dTy).real();
          gdelta[1] += 2.0 * (std::conj(g) * dTx).real();
        }
  }
}

static int row_of(const Model& m, int jb) { return m.batch_idx ? m.batch_idx[jb] : jb; }

extern "C" {

// ------------------------------------------------------------------------------------------
// forward + loss (O0..O6).  Outputs may be NULL.  Returns 0, -1 out of bounds.
// ------------------------------------------------------------------------------------------
int32_t orc_forward_loss(const orc_problem* p, const float* object, const float* probe,
                         const float* positions, const float* intensity, const int32_t* batch_idx,
                         double* loss, double* loss_per_pos, double* model_intensity) {
  Model m; model_init(m, p, object, probe, positions, intensity, batch_idx);
  const int J = p->n_batch; int err = 0;
  std::vector<double> Lj(J, 0.0);
#pragma omp parallel for schedule(dynamic)
  for (int jb = 0; jb < J; ++jb) {
    PosWork w; int jrow = row_of(m, jb);
    if (forward_pos(m, jrow, w) != 0) {
#pragma omp atomic write
      err = -1;
      continue;
    }
    if (model_intensity) for (long q = 0; q < m.NN; ++q) model_intensity[(long)jb * m.NN + q] = w.I[q];
    if (intensity) {
      double L = 0.0; const float* Iexp = intensity + (long)jrow * m.NN;
      for (long q = 0; q < m.NN; ++q) { double l, ww; orc_loss_pixel(p->loss, w.I[q], (double)Iexp[q], (double)p->loss_c, (double)p->eps, &l, &ww); L += l; }
      Lj[jb] = L;
    }
  }
  double L = 0.0; for (int jb = 0; jb < J; ++jb) { L += Lj[jb]; if (loss_per_pos) loss_per_pos[jb] = Lj[jb]; }
  if (loss) *loss = L;
  return err;
}

// ------------------------------------------------------------------------------------------
// loss + gradients (O0..O11) and the illumination map (O12).
//   grad_object [S][ony][onx] complex, grad_probe [M][N][N] complex   (dL/d conj(.))
//   grad_pos [J][2]  dL/dX per Angstrom (O10), illum [S][ony][onx] real — any may be NULL
// ------------------------------------------------------------------------------------------
int32_t orc_gradient(const orc_problem* p, const float* object, const float* probe,
                     const float* positions, const float* intensity, const int32_t* batch_idx,
                     double* grad_object, double* grad_probe, double* grad_pos, double* illum,
                     double* loss, double* loss_per_pos) {
  Model m; model_init(m, p, object, probe, positions, intensity, batch_idx);
  const int J = p->n_batch, N = m.N, M = m.M, S = m.S; const long NN = m.NN;
  const long on = (long)S * p->obj_ny * p->obj_nx;
  int err = 0;
  std::vector<double> Lj(J, 0.0);
  std::vector<cd> gO(on, cd(0.0)); std::vector<double> il(illum ? on : 0, 0.0);
  std::vector<std::vector<cd>> gPt(M, std::vector<cd>(NN, cd(0.0)));
#pragma omp parallel
  {
    std::vector<cd> gO_loc(on, cd(0.0)); std::vector<double> il_loc(illum ? on : 0, 0.0);
    std::vector<std::vector<cd>> gPt_loc(M, std::vector<cd>(NN, cd(0.0)));
#pragma omp for schedule(dynamic)
    for (int jb = 0; jb < J; ++jb) {
      PosWork w; int jrow = row_of(m, jb);
      if (forward_pos(m, jrow, w) != 0) {
#pragma omp atomic write
        err = -1;
        continue;
      }
      std::vector<std::vector<cd>> gT; double gd[2];
      adjoint_pos(m, jrow, w, &Lj[jb], gT, &gPt_loc, gd, false);
      const long os = (long)p->obj_ny * p->obj_nx;
      std::vector<cd> il_patch(illum ? NN : 0), il_slice(illum ? os : 0);
      for (int i = 0; i < S; ++i) {                                             // O8 last line: scatter-add
        if (illum) {                                                            // O12: sum_k |Psi_{i,k}|^2, scattered like gT_i
          for (long r = 0; r < NN; ++r) { double s = 0.0; for (int k = 0; k < M; ++k) s += std::norm(w.Psi[(long)i * M + k][r]); il_patch[r] = s; }
          std::fill(il_slice.begin(), il_slice.end(), cd(0.0));
        }
        if (p->shift_mode != 1) {
          scatter_add_window(N, p->obj_nx, gO_loc.data() + i * os, w.r0y, w.r0x, gT[i].data());
          if (illum) scatter_add_window(N, p->obj_nx, il_slice.data(), w.r0y, w.r0x, il_patch.data());
        } else {                                                                // bilinear mode: the same four weights
          scatter_add_window_bilinear(N, p->obj_nx, gO_loc.data() + i * os, w.r0y, w.r0x, w.dy, w.dx, gT[i].data());
          if (illum) scatter_add_window_bilinear(N, p->obj_nx, il_slice.data(), w.r0y, w.r0x, w.dy, w.dx, il_patch.data());
        }
        if (illum) for (long o = 0; o < os; ++o) il_loc[i * os + o] += il_slice[o].real();
      }
      if (grad_pos) { grad_pos[2 * jb + 0] = gd[0] / (double)p->pixel_size; grad_pos[2 * jb + 1] = gd[1] / (double)p->pixel_size; }
    }
#pragma omp critical
    {
      for (long o = 0; o < on; ++o) gO[o] += gO_loc[o];
      if (illum) for (long o = 0; o < on; ++o) il[o] += il_loc[o];
      for (int k = 0; k < M; ++k) for (long q = 0; q < NN; ++q) gPt[k][q] += gPt_loc[k][q];
    }
  }
  if (grad_object) for (long o = 0; o < on; ++o) { grad_object[2 * o] = gO[o].real(); grad_object[2 * o + 1] = gO[o].imag(); }
  if (illum) for (long o = 0; o < on; ++o) illum[o] = il[o];
  if (grad_probe)
    for (int k = 0; k < M; ++k) {                                               // O11
      Finv2(N, gPt[k].data());
      for (long r = 0; r < NN; ++r) { grad_probe[2 * (k * NN + r)] = gPt[k][r].real(); grad_probe[2 * (k * NN + r) + 1] = gPt[k][r].imag(); }
    }
  double L = 0.0; for (int jb = 0; jb < J; ++jb) { L += Lj[jb]; if (loss_per_pos) loss_per_pos[jb] = Lj[jb]; }
  if (loss) *loss = L;
  return err;
}

// ------------------------------------------------------------------------------------------
// O13/O14: LSQML-style step-size terms, second sweep over the batch.
//   grad_object/grad_probe: the batch-aggregated gradients (double, as returned by orc_gradient)
//   illum_prev: [S][ony][onx] running probe-intensity sum of the previous iteration
//   step_terms: [J][2S+6]:  (numO,denO) per slice, (numP,denP), (numX_y,denX_y), (numX_x,denX_x)
// chi_{i,k} := -c gPhi_{i,k}, c = lsqml_chi_scale: steepest-descent wavefront update (c = 1, reading R20) or the
// modulus-constraint update of PAPER.md:173 (c = 2, reading R31); the directions dOhat, dPhat are built from the same chi
// (PAPER.md:213-219), so they carry the factor c too.
// Bilinear mode (readings R1, R30): the patch of dOhat is the same four-tap sample as the patch of O; the position enters through
// the patches of every slice, so numX_a = sum_{i,k,r} Re[chi_{i,k} conj(Psi_{i,k} dT_i/df_a)], denX_a = sum_{i,k,r} |Psi_{i,k} dT_i/df_a|^2
// (f in px), the least-squares step of the exit waves' first-order change, slice by slice as PAPER.md:221 does for the object.
// ------------------------------------------------------------------------------------------
int32_t orc_step_terms(const orc_problem* p, const float* object, const float* probe,
                       const float* positions, const float* intensity, const int32_t* batch_idx,
                       const double* grad_object, const double* grad_probe, const double* illum_prev,
                       const double* probe_precond /* [N][N] or NULL: constant 1 (R19), reading R25 */,
                       double* step_terms) {
  if (p->lsqml_chi_scale != 1.0f && p->loss != 0) return -2;                    // PAPER.md:173 gives the update for the amplitude model
  Model m; model_init(m, p, object, probe, positions, intensity, batch_idx);
  const int J = p->n_batch, N = m.N, M = m.M, S = m.S; const long NN = m.NN;
  const long on = (long)S * p->obj_ny * p->obj_nx, os = (long)p->obj_ny * p->obj_nx;
  const double cs = (double)p->lsqml_chi_scale;
  const bool bil = p->shift_mode == 1;
  std::vector<cd> dOhat(on);
  for (long o = 0; o < on; ++o)                                                 // O13
    dOhat[o] = -cs * cd(grad_object[2 * o], grad_object[2 * o + 1]) / (illum_prev[o] + (double)p->lsqml_delta_o);
  std::vector<std::vector<cd>> dPhat_t(M, std::vector<cd>(NN));                 // F(dPhat_k)
  for (int k = 0; k < M; ++k) {
    for (long r = 0; r < NN; ++r)
      dPhat_t[k][r] = -cs * cd(grad_probe[2 * (k * NN + r)], grad_probe[2 * (k * NN + r) + 1]) / ((probe_precond ? probe_precond[r] : 1.0) + (double)p->lsqml_delta_p);
    F2(N, dPhat_t[k].data());
  }
  int err = 0; const int W = 2 * S + 6;
#pragma omp parallel for schedule(dynamic)
  for (int jb = 0; jb < J; ++jb) {
    PosWork w; int jrow = row_of(m, jb);
    if (forward_pos(m, jrow, w) != 0) {
#pragma omp atomic write
      err = -1;
      continue;
    }
    std::vector<std::vector<cd>> gT; double gd[2], Lj;
    adjoint_pos(m, jrow, w, &Lj, gT, nullptr, gd, true);
    double* out = step_terms + (long)jb * W;
    double numP = 0, denP = 0, numX[2] = {0, 0}, denX[2] = {0, 0};
    for (int i = 0; i < S; ++i) {                                               // O14 object
      double num = 0.0, den = 0.0;
      std::vector<cd> dOp(NN);                                                  // dOhat_i in the probe view: the patch, sampled like T_i
      if (!bil) gather_window(N, p->obj_nx, dOhat.data() + i * os, w.r0y, w.r0x, dOp.data());
      else gather_window_bilinear(N, p->obj_nx, dOhat.data() + i * os, w.r0y, w.r0x, w.dy, w.dx, dOp.data());
      for (int k = 0; k < M; ++k)
        for (long r = 0; r < NN; ++r) {
          cd u = dOp[r] * w.Psi[(long)i * M + k][r];
          cd chi = -cs * w.gPhi[(long)i * M + k][r];
          num += (chi * std::conj(u)).real(); den += std::norm(u);
        }
      out[2 * i] = num; out[2 * i + 1] = den;
      if (bil)                                                                  // position terms through the patch (R30)
        for (int y = 0; y < N; ++y)
          for (int x = 0; x < N; ++x) {
            auto O = [&](int dy, int dx) { return m.obj[((long)i * p->obj_ny + (w.r0y + y + dy)) * p->obj_nx + (w.r0x + x + dx)]; };
            const cd dT[2] = {bil_w(0, w.dx) * (O(1, 0) - O(0, 0)) + bil_w(1, w.dx) * (O(1, 1) - O(0, 1)),
                              bil_w(0, w.dy) * (O(0, 1) - O(0, 0)) + bil_w(1, w.dy) * (O(1, 1) - O(1, 0))};
            const long r = (long)y * N + x;
            for (int k = 0; k < M; ++k)
              for (int a = 0; a < 2; ++a) {
                cd ss = w.Psi[(long)i * M + k][r] * dT[a]; cd chi = -cs * w.gPhi[(long)i * M + k][r];
                numX[a] += (chi * std::conj(ss)).real(); denX[a] += std::norm(ss);
              }
          }
    }
    for (int k = 0; k < M; ++k) {
      std::vector<cd> v(NN);
      for (long q = 0; q < NN; ++q) v[q] = w.R[q] * dPhat_t[k][q];              // shift_j(dPhat_k)
      Finv2(N, v.data());
      for (long r = 0; r < NN; ++r) {
        cd vv = v[r] * w.T[0][r]; cd chi = -cs * w.gPhi[k][r];                  // slice 0: index 0*M+k
        numP += (chi * std::conj(vv)).real(); denP += std::norm(vv);
      }
      for (int a = 0; a < 2 && !bil; ++a) {
        std::vector<cd> s(NN);
        for (int qy = 0; qy < N; ++qy)
          for (int qx = 0; qx < N; ++qx) {
            long q = (long)qy * N + qx; double fa = (a == 0) ? freq(qy, N) : freq(qx, N);
            s[q] = cd(0.0, -2.0 * PI * fa) * w.R[q] * m.Pt[k][q];               // d Psi_0 / d delta_a, Fourier side
          }
        Finv2(N, s.data());
        for (long r = 0; r < NN; ++r) {
          cd ss = s[r] * w.T[0][r]; cd chi = -cs * w.gPhi[k][r];
          numX[a] += (chi * std::conj(ss)).real(); denX[a] += std::norm(ss);
        }
      }
    }
    out[2 * S + 0] = numP; out[2 * S + 1] = denP;
    out[2 * S + 2] = numX[0]; out[2 * S + 3] = denX[0];
    out[2 * S + 4] = numX[1]; out[2 * S + 5] = denX[1];
  }
  return err;
}

// ------------------------------------------------------------------------------------------
// O15 / H15 update.  mode 0: SGD z <- z - lr g.  mode 1: LSQML-style (R18):
//   alpha_{O,i} = sum_j numO / (sum_j denO + gamma);  O_i += beta_O alpha_{O,i} dOhat_i   etc.
// object/probe/positions are double in/out here (the test converts); positions rows batch_idx only.
// ------------------------------------------------------------------------------------------
int32_t orc_apply_update(const orc_problem* p, int32_t mode, double* object, double* probe, double* positions,
                         const double* grad_object, const double* grad_probe, const double* grad_pos,
                         const double* illum_prev, const double* step_terms, const int32_t* batch_idx,
                         double lr_obj, double lr_probe, double lr_pos, double beta_obj, double beta_probe,
                         double gamma, const double* probe_precond /* [N][N] or NULL, as in orc_step_terms */) {
  const int J = p->n_batch, M = p->n_modes, S = p->n_slices; const long NN = (long)p->n * p->n;
  const long os = (long)p->obj_ny * p->obj_nx;
  if (mode == 0) {
    if (object && grad_object) for (long o = 0; o < 2 * S * os; ++o) object[o] -= lr_obj * grad_object[o];
    if (probe && grad_probe) for (long r = 0; r < 2 * M * NN; ++r) probe[r] -= lr_probe * grad_probe[r];
    if (positions && grad_pos)
      for (int jb = 0; jb < J; ++jb) { int row = batch_idx ? batch_idx[jb] : jb;
        positions[2 * row] -= lr_pos * grad_pos[2 * jb]; positions[2 * row + 1] -= lr_pos * grad_pos[2 * jb + 1]; }
    return 0;
  }
  const int W = 2 * S + 6;
  const double cs = (double)p->lsqml_chi_scale;
  if (object && grad_object)
    for (int i = 0; i < S; ++i) {
      double num = 0, den = 0;
      for (int jb = 0; jb < J; ++jb) { num += step_terms[(long)jb * W + 2 * i]; den += step_terms[(long)jb * W + 2 * i + 1]; }
      double alpha = num / (den + gamma);
      for (long o = 0; o < os; ++o) {
        long g = (long)i * os + o; double d = illum_prev[g] + (double)p->lsqml_delta_o;
        object[2 * g] += beta_obj * alpha * (-cs * grad_object[2 * g] / d);      // dOhat = -c gO / d (O13)
        object[2 * g + 1] += beta_obj * alpha * (-cs * grad_object[2 * g + 1] / d);
      }
    }
  if (probe && grad_probe) {
    double num = 0, den = 0;
    for (int jb = 0; jb < J; ++jb) { num += step_terms[(long)jb * W + 2 * S]; den += step_terms[(long)jb * W + 2 * S + 1]; }
    double alpha = num / (den + gamma);
    for (long r = 0; r < 2 * M * NN; ++r)
      probe[r] += beta_probe * alpha * (-cs * grad_probe[r] / ((probe_precond ? probe_precond[(r / 2) % NN] : 1.0) + (double)p->lsqml_delta_p));
  }
  if (positions)
    for (int jb = 0; jb < J; ++jb) { int row = batch_idx ? batch_idx[jb] : jb;
      for (int a = 0; a < 2; ++a) {
        double num = step_terms[(long)jb * W + 2 * S + 2 + 2 * a], den = step_terms[(long)jb * W + 2 * S + 3 + 2 * a];
        positions[2 * row + a] += (double)p->pixel_size * num / (den + gamma);
      } }
  return 0;
}

// ------------------------------------------------------------------------------------------
// LSQML probe preconditioner (reading R25): "the summed object intensity sum prod_i |O_i|^2 is recorded in
// the probe/cutout view": objtrans[r] = sum_{j in group} prod_i |O_i[r0_j + r]|^2, r in the N x N window.  The caller
// keeps the running sum over an iteration and hands last iteration's total back as probe_precond (like illum_prev).
// ------------------------------------------------------------------------------------------
int32_t orc_object_transparency(const orc_problem* p, const float* object, const float* positions, const int32_t* batch_idx,
                                double* objtrans /* [N][N] */) {
  const int N = p->n, S = p->n_slices, J = p->n_batch;
  for (long r = 0; r < (long)N * N; ++r) objtrans[r] = 0.0;
  for (int jb = 0; jb < J; ++jb) {
    const int jrow = batch_idx ? batch_idx[jb] : jb;
    int32_t r0y, r0x; float dy, dx;
    orc_position_split(positions[2 * jrow + 0], p->pixel_size, N, &r0y, &dy);
    orc_position_split(positions[2 * jrow + 1], p->pixel_size, N, &r0x, &dx);
    if (r0y < 0 || r0x < 0 || r0y + N > p->obj_ny || r0x + N > p->obj_nx) return -1;
    for (int y = 0; y < N; ++y)
      for (int x = 0; x < N; ++x) {
        double t = 1.0;
        for (int i = 0; i < S; ++i) {
          const long o = ((long)i * p->obj_ny + (r0y + y)) * p->obj_nx + (r0x + x);
          t *= (double)object[2 * o] * object[2 * o] + (double)object[2 * o + 1] * object[2 * o + 1];
        }
        objtrans[(long)y * N + x] += t;
      }
  }
  return 0;
}

// ------------------------------------------------------------------------------------------
// LSQML final slice update with PER-POSITION step sizes, exactly as printed at PAPER.md:225 (reading R24):
//   alpha_{O,i,j} = numO[j,i] / (denO[j,i] + gamma)                       (sums over r and k only)
//   W_i[r]  = sum_{j in group} alpha_{O,i,j} sum_k |Psi_{i,k,j}[r - r0_j]|^2   (numerator weight of :225)
//   I_i[r]  = sum_{j in group} sum_k |Psi_{i,k,j}[r - r0_j]|^2                 (denominator of :225 = O12 of this batch)
//   O_i[r] += beta_O dOhat_i[r] W_i[r] / I_i[r]      where I_i[r] > 0 ; pixels no window of the group covers are left alone
// dOhat_i does not depend on j, so it leaves the group sum.  orc_weighted_illum returns W; the update is below.
// ------------------------------------------------------------------------------------------
int32_t orc_weighted_illum(const orc_problem* p, const float* object, const float* probe, const float* positions,
                           const int32_t* batch_idx, const double* step_terms, double gamma, double* willum) {
  if (p->shift_mode == 1) return -2;
  Model m; model_init(m, p, object, probe, positions, nullptr, batch_idx);
  const int J = p->n_batch, N = m.N, M = m.M, S = m.S; const int W = 2 * S + 6;
  const long on = (long)S * p->obj_ny * p->obj_nx;
  for (long o = 0; o < on; ++o) willum[o] = 0.0;
  for (int jb = 0; jb < J; ++jb) {                                              // plain serial loop: fixed summation order
    PosWork w; int jrow = row_of(m, jb);
    if (forward_pos(m, jrow, w) != 0) return -1;
    for (int i = 0; i < S; ++i) {
      const double alpha = step_terms[(long)jb * W + 2 * i] / (step_terms[(long)jb * W + 2 * i + 1] + gamma);
      for (int y = 0; y < N; ++y)
        for (int x = 0; x < N; ++x) {
          double s = 0.0;
          for (int k = 0; k < M; ++k) s += std::norm(w.Psi[(long)i * M + k][(long)y * N + x]);
          willum[((long)i * p->obj_ny + (w.r0y + y)) * p->obj_nx + (w.r0x + x)] += alpha * s;
        }
    }
  }
  return 0;
}

// object (double complex, in/out) += beta_O dOhat W / I, dOhat = -gO / (illum_prev + delta_O)
int32_t orc_lsqml_weighted_object(const orc_problem* p, double* object, const double* grad_object, const double* illum_prev,
                                  const double* illum_batch, const double* willum, double beta_obj) {
  const long on = (long)p->n_slices * p->obj_ny * p->obj_nx;
  for (long o = 0; o < on; ++o) {
    if (!(illum_batch[o] > 0.0)) continue;
    const double f = (double)p->lsqml_chi_scale * beta_obj * (willum[o] / illum_batch[o]) / (illum_prev[o] + (double)p->lsqml_delta_o);
    object[2 * o] += f * (-grad_object[2 * o]);
    object[2 * o + 1] += f * (-grad_object[2 * o + 1]);
  }
  return 0;
}

// ------------------------------------------------------------------------------------------
// Multislice ePIE ("3PIE") update directions for one group of positions (reading R23).
//   detector:  chi~_k = ( sqrt(Iexp+c) / (eps + sqrt(I+c)) - 1 ) psi~_k            (amplitude model only;
//              c = 0 is the classic modulus constraint)
//   exit:      chi_{S-1,k} = N Finv(chi~_k)                                          (psi~ = F(.)/N, reading R5)
//   slice i:   dO_{i,k}   = conj(Psi_{i,k}) / max_r |Psi_{i,k}|^2 . chi_{i,k}        (P_i = entering wave)
//              chi'_{i,k} = conj(T_i)      / max_r |T_i|^2       . chi_{i,k}        (max over the window)
//              chi_{i-1,k} = Finv( conj(H_{i-1}) F(chi'_{i,k}) )                     ("propagated backwards")
//   object direction  dO_i[r0 + r] += sum_k dO_{i,k}[r], summed over the group
//   probe direction   dP_k = (1/J) sum_j shift_j^{-1}( chi'_{0,k,j} )                ("averaged across the group")
// The caller applies O_i += beta_object dO_i, P_k += beta_probe dP_k.  Fourier-shift mode and amplitude loss only
// (returns -2 otherwise).  dir_object [S][ony][onx], dir_probe [M][N][N] complex (doubles).
// ------------------------------------------------------------------------------------------
int32_t orc_epie(const orc_problem* p, const float* object, const float* probe, const float* positions,
                 const float* intensity, const int32_t* batch_idx, double* dir_object, double* dir_probe,
                 double* loss, double* loss_per_pos) {
  if (p->loss != 0 || p->shift_mode != 0) return -2;
  Model m; model_init(m, p, object, probe, positions, intensity, batch_idx);
  const int J = p->n_batch, N = m.N, M = m.M, S = m.S; const long NN = m.NN;
  const long on = (long)S * p->obj_ny * p->obj_nx;
  std::vector<cd> dO(on, cd(0.0));
  std::vector<std::vector<cd>> dPt(M, std::vector<cd>(NN, cd(0.0)));           // sum_j conj(R_j) F(chi'_0), Fourier side
  double L = 0.0; int err = 0;
  for (int jb = 0; jb < J; ++jb) {                                             // plain loop: fixed summation order
    PosWork w; int jrow = row_of(m, jb);
    if (forward_pos(m, jrow, w) != 0) { err = -1; continue; }
    const float* Iexp = intensity + (long)jrow * NN;
    std::vector<double> u(NN); double Lj = 0.0;
    for (long q = 0; q < NN; ++q) {
      double a = std::sqrt(w.I[q] + (double)p->loss_c), ae = std::sqrt((double)Iexp[q] + (double)p->loss_c);
      Lj += 0.5 * (a - ae) * (a - ae);
      u[q] = ae / ((double)p->eps + a) - 1.0;
    }
    L += Lj; if (loss_per_pos) loss_per_pos[jb] = Lj;
    std::vector<double> tmax(S, 0.0);
    for (int i = 0; i < S; ++i) for (long r = 0; r < NN; ++r) tmax[i] = std::max(tmax[i], std::norm(w.T[i][r]));
    for (int k = 0; k < M; ++k) {
      std::vector<cd> chi(NN);
      for (long q = 0; q < NN; ++q) chi[q] = u[q] * w.psit[k][q];
      Finv2(N, chi.data());
      for (long r = 0; r < NN; ++r) chi[r] *= (double)N;
      for (int i = S - 1; i >= 0; --i) {
        const std::vector<cd>& Psi = w.Psi[(long)i * M + k];
        double pmax = 0.0; for (long r = 0; r < NN; ++r) pmax = std::max(pmax, std::norm(Psi[r]));
        // PAPER.md:203 divides by max|Psi|^2; an identically zero wave (an unused probe mode) gives 0/0 there.  Reading R23b
        // (DESIGN.md §3): such a wave contributes nothing, i.e. 1/max is taken as 0; likewise 1/max|T|^2 for an opaque window.
        const double ipmax = pmax > 0.0 ? 1.0 / pmax : 0.0, itmax = tmax[i] > 0.0 ? 1.0 / tmax[i] : 0.0;
        for (int y = 0; y < N; ++y)
          for (int x = 0; x < N; ++x) {
            long r = (long)y * N + x;
            dO[((long)i * p->obj_ny + (w.r0y + y)) * p->obj_nx + (w.r0x + x)] += std::conj(Psi[r]) * ipmax * chi[r];
          }
        for (long r = 0; r < NN; ++r) chi[r] = std::conj(w.T[i][r]) * itmax * chi[r];
        if (i > 0) {
          F2(N, chi.data());
          for (long q = 0; q < NN; ++q) chi[q] *= std::conj(m.H[i - 1][q]);
          Finv2(N, chi.data());
        }
      }
      F2(N, chi.data());                                                       // undo the sub-pixel shift on the Fourier side
      for (long q = 0; q < NN; ++q) dPt[k][q] += std::conj(w.R[q]) * chi[q];
    }
  }
  if (dir_object) for (long o = 0; o < on; ++o) { dir_object[2 * o] = dO[o].real(); dir_object[2 * o + 1] = dO[o].imag(); }
  if (dir_probe)
    for (int k = 0; k < M; ++k) {
      Finv2(N, dPt[k].data());
      for (long r = 0; r < NN; ++r) { dir_probe[2 * (k * NN + r)] = dPt[k][r].real() / J; dir_probe[2 * (k * NN + r) + 1] = dPt[k][r].imag() / J; }
    }
  if (loss) *loss = L;
  return err;
}

// ------------------------------------------------------------------------------------------
// Cost regularisers (the paper lists them by name only — reading R26).  field is [S][ny][nx] complex
// (object slices, or probe modes with S = M); returns R and ADDS dR/dconj(field) into grad (dR = 2 Re sum conj(g) dz).
//   kind 0  L2            R = w sum |z - ref|^2                      ("penalizes ... a non-vacuum object": ref = 1; probe: ref = 0)
//   kind 1  L1            R = w sum sqrt(|z - ref|^2 + eps^2)       (smoothed modulus)
//   kind 2  Tikhonov      R = w sum_{d in x,y} sum |D_d z|^2        (forward differences inside a slice, no wrap-around)
//   kind 3  TV            R = w sum_{d in x,y} sum sqrt(|D_d z|^2 + eps^2)
//   kind 4  layer Tikhonov, kind 5 layer TV: the same with the one difference along the depth axis, D_z z = z_{i+1} - z_i
//   kind 6  L1 on the object PHASE ("L1 regularization: (object, object phase, ...)"; reading R26b):
//           R = w sum sqrt(phi^2 + eps^2), phi = arg z in (-pi, pi] (principal value: object slices are weak phase objects,
//           |phi| << pi).  With phi = Im log z, d phi / d conj(z) = i z / (2 |z|^2), hence
//           dR/dconj(z) = w phi / sqrt(phi^2 + eps^2) * i z / (2 |z|^2); a zero pixel, and phi = 0 with eps = 0, contribute no gradient
//   kind 7  L1 on the object's Fourier amplitudes per slice ("object power spectrum ... to bias the reconstruction towards
//           periodic solutions"; reading R26c: the L1 norm of the power spectrum |Z|^2 itself is N times the L2 regulariser by Parseval, so
//           the sparsity-promoting form is the L1 norm of its square root): R = w sum_s sum_q sqrt(|Z_s[q]|^2 + eps^2); ref unused
// ------------------------------------------------------------------------------------------
static double reg_phi(int tv, double a2, double eps) { return tv ? std::sqrt(a2 + eps * eps) : a2; }
static double reg_dphi(int tv, double a2, double eps) { return tv ? 0.5 / std::sqrt(a2 + eps * eps) : 1.0; }   // d phi / d(a2)

double orc_cost_regularizer(int32_t kind, double weight, double ref, double eps, int32_t S, int32_t ny, int32_t nx,
                            const double* field, double* grad) {
  const long os = (long)ny * nx, n = (long)S * os;
  auto Z = [&](long i) { return cd(field[2 * i], field[2 * i + 1]); };
  auto addg = [&](long i, cd v) { grad[2 * i] += v.real(); grad[2 * i + 1] += v.imag(); };
  double R = 0.0;
  if (kind == 0 || kind == 1) {
    for (long i = 0; i < n; ++i) {
      cd u = Z(i) - ref; double a2 = std::norm(u);
      R += weight * reg_phi(kind == 1, a2, eps);
      addg(i, weight * reg_dphi(kind == 1, a2, eps) * u);              // d phi(|u|^2) / d conj(z) = phi' u
    }
    return R;
  }
  if (kind == 6) {
    for (long i = 0; i < n; ++i) {
      const cd z = Z(i); const double a2 = std::norm(z);
      if (a2 == 0.0) continue;
      const double phi = std::atan2(z.imag(), z.real()), q = std::sqrt(phi * phi + eps * eps);
      R += weight * q;
      if (q > 0.0) addg(i, weight * (phi / q) * cd(0.0, 1.0) * z / (2.0 * a2));
    }
    return R;
  }
  if (kind == 7) {
    // R = w sum_s sum_q sqrt(|Z_s[q]|^2 + eps^2), Z_s = F z_s the unnormalised 2-D DFT of slice s over the whole (ny x nx) slice,
    // any size: rows, then columns, by the definition (twiddle index reduced mod the length exactly).
    // dR/dconj(Z) = w Z / (2 sqrt(|Z|^2 + eps^2)) and Z is linear in z, so dR/dconj(z) = F^H (dR/dconj(Z)).
    std::vector<cd> wx(nx), wy(ny);
    for (int m = 0; m < nx; ++m) wx[m] = std::polar(1.0, -2.0 * M_PI * m / nx);
    for (int m = 0; m < ny; ++m) wy[m] = std::polar(1.0, -2.0 * M_PI * m / ny);
    std::vector<cd> A(os), Zq(os);
    for (int s = 0; s < S; ++s) {
      for (int y = 0; y < ny; ++y)
        for (int kx = 0; kx < nx; ++kx) {
          cd a = 0.0;
          for (int x = 0; x < nx; ++x) a += Z((long)s * os + (long)y * nx + x) * wx[(long)x * kx % nx];
          A[(long)y * nx + kx] = a;
        }
      for (int ky = 0; ky < ny; ++ky)
        for (int kx = 0; kx < nx; ++kx) {
          cd a = 0.0;
          for (int y = 0; y < ny; ++y) a += A[(long)y * nx + kx] * wy[(long)y * ky % ny];
          Zq[(long)ky * nx + kx] = a;
        }
      for (long q = 0; q < os; ++q) {
        const double a2 = std::norm(Zq[q]), r = std::sqrt(a2 + eps * eps);
        R += weight * r;
        Zq[q] = r > 0.0 ? weight * Zq[q] / (2.0 * r) : cd(0.0);     // dR/dconj(Z); |Z| = 0 with eps = 0: subgradient 0
      }
      if (!grad) continue;
      for (int y = 0; y < ny; ++y)                                    // F^H: conjugate kernels, columns then rows
        for (int kx = 0; kx < nx; ++kx) {
          cd a = 0.0;
          for (int ky = 0; ky < ny; ++ky) a += Zq[(long)ky * nx + kx] * std::conj(wy[(long)y * ky % ny]);
          A[(long)y * nx + kx] = a;
        }
      for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
          cd a = 0.0;
          for (int kx = 0; kx < nx; ++kx) a += A[(long)y * nx + kx] * std::conj(wx[(long)x * kx % nx]);
          addg((long)s * os + (long)y * nx + x, a);
        }
    }
    return R;
  }
  const int tv = (kind == 3 || kind == 5);
  const long strides[3] = {1, (long)nx, os};
  for (int d = 0; d < 3; ++d) {
    if ((kind == 2 || kind == 3) && d == 2) continue;                  // in-plane kinds: x and y only
    if ((kind == 4 || kind == 5) && d != 2) continue;                  // layer kinds: depth only
    for (int s = 0; s < S; ++s)
      for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
          if ((d == 0 && x + 1 >= nx) || (d == 1 && y + 1 >= ny) || (d == 2 && s + 1 >= S)) continue;
          long i = (long)s * os + (long)y * nx + x, j = i + strides[d];
          cd u = Z(j) - Z(i); double a2 = std::norm(u);
          R += weight * reg_phi(tv, a2, eps);
          cd c = weight * reg_dphi(tv, a2, eps) * u;
          addg(j, c); addg(i, -c);
        }
  }
  return R;
}

// ------------------------------------------------------------------------------------------
// Constraint regularisers (reading R27).  field [S][ny][nx] complex, in place.
//   kind 0  amplitude clamp: |z| limited to [a, b], phase kept (a zero pixel with a > 0 becomes the real number a)
//   kind 1  support mask:    z[s][y][x] *= mask[y][x]   (probe support in real space; mask [ny][nx] real)
//   kind 2  layer blur:      Gaussian blur along the depth axis, sigma = a slices, REAL-SPACE convolution (the paper's
//                            reason: no bleeding from top to bottom through periodic boundaries): out[p] = sum_t w_t z[p+t] /
//                            sum_t w_t over the taps |t| <= ceil(4 sigma) that fall inside, w_t = exp(-t^2 / (2 sigma^2))
//   kind 3  object low pass: the same blur along x then along y, sigma = a px
//   kind 4  probe support in reciprocal space, kind 5 object phase deramp: see the code below
// ------------------------------------------------------------------------------------------
static void blur_axis(int S, int ny, int nx, int axis, double sigma, std::vector<cd>& z) {
  const int R = (int)std::ceil(4.0 * sigma);
  const long os = (long)ny * nx; const long stride = axis == 0 ? 1 : axis == 1 ? nx : os;
  const int len = axis == 0 ? nx : axis == 1 ? ny : S;
  std::vector<cd> out(z.size());
  for (int s = 0; s < S; ++s)
    for (int y = 0; y < ny; ++y)
      for (int x = 0; x < nx; ++x) {
        const long i = (long)s * os + (long)y * nx + x; const int c = axis == 0 ? x : axis == 1 ? y : s;
        cd acc = 0.0; double wsum = 0.0;
        for (int t = -R; t <= R; ++t) {
          if (c + t < 0 || c + t >= len) continue;
          double w = std::exp(-(double)t * t / (2.0 * sigma * sigma));
          acc += w * z[i + (long)t * stride]; wsum += w;
        }
        out[i] = acc / wsum;
      }
  z.swap(out);
}

int32_t orc_apply_constraint(int32_t kind, double a, double b, const double* mask, int32_t S, int32_t ny, int32_t nx, double* field) {
  const long os = (long)ny * nx, n = (long)S * os;
  if (kind == 0) {
    for (long i = 0; i < n; ++i) {
      cd z(field[2 * i], field[2 * i + 1]); double m = std::abs(z);
      double t = m < a ? a : (m > b ? b : m);
      if (t == m) continue;
      cd u = m > 0.0 ? z / m : cd(1.0, 0.0);
      field[2 * i] = t * u.real(); field[2 * i + 1] = t * u.imag();
    }
    return 0;
  }
  if (kind == 1) {
    for (long i = 0; i < n; ++i) { field[2 * i] *= mask[i % os]; field[2 * i + 1] *= mask[i % os]; }
    return 0;
  }
  if (kind == 4) {
    // probe support in RECIPROCAL space: z <- Finv(mask .* F(z)), mask [n][n] real, zero frequency at [0][0]
    if (ny != nx) return -3;
    std::vector<cd> f(os);
    for (int s = 0; s < S; ++s) {
      for (long r = 0; r < os; ++r) f[r] = cd(field[2 * (s * os + r)], field[2 * (s * os + r) + 1]);
      F2(nx, f.data());
      for (long q = 0; q < os; ++q) f[q] *= mask[q];
      Finv2(nx, f.data());
      for (long r = 0; r < os; ++r) { field[2 * (s * os + r)] = f[r].real(); field[2 * (s * os + r) + 1] = f[r].imag(); }
    }
    return 0;
  }
  if (kind == 5) {
    // object phase deramp ("removes an affine phase ramp from the object"; reading R29, no phase unwrapping):
    // per slice, slopes from the amplitude-weighted mean phase step b = arg sum z[y+1,x] conj(z[y,x]), c likewise along x;
    // offset a = arg sum z exp(-i(b (y - yc) + c (x - xc))) about the centre; z <- z exp(-i(a + b (y - yc) + c (x - xc)))
    const double yc = 0.5 * (ny - 1), xc = 0.5 * (nx - 1);
    for (int s = 0; s < S; ++s) {
      auto Zs = [&](int y, int x) { long i = (long)s * os + (long)y * nx + x; return cd(field[2 * i], field[2 * i + 1]); };
      cd sy = 0.0, sx = 0.0, sa = 0.0;
      for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
          if (y + 1 < ny) sy += Zs(y + 1, x) * std::conj(Zs(y, x));
          if (x + 1 < nx) sx += Zs(y, x + 1) * std::conj(Zs(y, x));
        }
      const double bb = std::arg(sy), cc = std::arg(sx);
      for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) sa += Zs(y, x) * std::polar(1.0, -(bb * (y - yc) + cc * (x - xc)));
      const double aa = std::arg(sa);
      for (int y = 0; y < ny; ++y)
        for (int x = 0; x < nx; ++x) {
          cd v = Zs(y, x) * std::polar(1.0, -(aa + bb * (y - yc) + cc * (x - xc)));
          long i = (long)s * os + (long)y * nx + x; field[2 * i] = v.real(); field[2 * i + 1] = v.imag();
        }
    }
    return 0;
  }
  if (!(a > 0.0)) return -3;
  std::vector<cd> z(n);
  for (long i = 0; i < n; ++i) z[i] = cd(field[2 * i], field[2 * i + 1]);
  if (kind == 2) blur_axis(S, ny, nx, 2, a, z);
  else if (kind == 3) { blur_axis(S, ny, nx, 0, a, z); blur_axis(S, ny, nx, 1, a, z); }
  else return -3;
  for (long i = 0; i < n; ++i) { field[2 * i] = z[i].real(); field[2 * i + 1] = z[i].imag(); }
  return 0;
}

// ------------------------------------------------------------------------------------------
// Adam ("SGD, Adam and its variants [62, 63]"; Kingma & Ba's algorithm 1; reading R28: for a complex variable
// the first moment is complex and the second moment uses |g|^2, the complex-safe form of the library the paper names).
//   m <- b1 m + (1 - b1) g ;  v <- b2 v + (1 - b2) |g|^2 ;  z <- z - lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps)
// is_complex = 0: n real numbers (positions), |g|^2 = g^2.
// ------------------------------------------------------------------------------------------
int32_t orc_adam_update(int32_t is_complex, double* z, const double* g, double* m, double* v, int64_t n, double lr, double b1,
                        double b2, double eps, int32_t t) {
  const double c1 = 1.0 - std::pow(b1, (double)t), c2 = 1.0 - std::pow(b2, (double)t);
  for (int64_t i = 0; i < n; ++i) {
    if (is_complex) {
      m[2 * i] = b1 * m[2 * i] + (1.0 - b1) * g[2 * i]; m[2 * i + 1] = b1 * m[2 * i + 1] + (1.0 - b1) * g[2 * i + 1];
      v[i] = b2 * v[i] + (1.0 - b2) * (g[2 * i] * g[2 * i] + g[2 * i + 1] * g[2 * i + 1]);
      const double d = std::sqrt(v[i] / c2) + eps;
      z[2 * i] -= lr * (m[2 * i] / c1) / d; z[2 * i + 1] -= lr * (m[2 * i + 1] / c1) / d;
    } else {
      m[i] = b1 * m[i] + (1.0 - b1) * g[i];
      v[i] = b2 * v[i] + (1.0 - b2) * g[i] * g[i];
      z[i] -= lr * (m[i] / c1) / (std::sqrt(v[i] / c2) + eps);
    }
  }
  return 0;
}

int32_t orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
