// regularizers.cuh — SURVEY §8(f) rank 3: cost regularisers (reading R26), constraint regularisers
// (R27) and the Adam update (R28).  Object-sized elementwise / stencil kernels, HBM-bound:
// one read of the field (+ neighbours from L1/L2) and one read-modify-write of the gradient per call.  Included at the end of
// ptycho_kernels.cu (it uses that file's launch accounting); the C ABI is declared in include/ptycho.h.
// Owner-computes everywhere (no atomics); the cost is a fixed-grid, fixed-order fp64 sum, so results are bitwise reproducible.
#pragma once

namespace {

constexpr int kRegBlocks = 1024, kRegThreads = 256;

__device__ __forceinline__ float reg_phi(bool tv, float a2, float eps2) { return tv ? sqrtf(a2 + eps2) : a2; }
__device__ __forceinline__ float reg_dphi(bool tv, float a2, float eps2) { return tv ? 0.5f * rsqrtf(a2 + eps2) : 1.0f; }

// kinds L2 / L1: pointwise
__global__ void __launch_bounds__(kRegThreads) k_reg_point(int l1, float w, float ref, float eps2, size_t n, const cf* z, cf* g, double* part) {
  __shared__ double red[kRegThreads / 32];
  double acc[1] = {0.0};
  for (size_t i = (size_t)blockIdx.x * kRegThreads + threadIdx.x; i < n; i += (size_t)kRegBlocks * kRegThreads) {
    const cf u = make_float2(z[i].x - ref, z[i].y);
    const float a2 = fmaf(u.x, u.x, u.y * u.y);
    if (l1 && a2 + eps2 == 0.f) continue;                            // |0| with eps = 0: subgradient 0
    acc[0] += (double)(w * reg_phi(l1, a2, eps2));
    if (g) { const float c = w * reg_dphi(l1, a2, eps2); g[i] = make_float2(fmaf(c, u.x, g[i].x), fmaf(c, u.y, g[i].y)); }
  }
  block_sum<kRegThreads, 1>(acc, red);
  if (threadIdx.x == 0) part[blockIdx.x] = acc[0];
}

// kind L1 on the phase (reading R26b): R = w sum sqrt(phi^2 + eps^2), phi = arg z ; dR/dconj(z) = w phi / sqrt(.) * i z / (2 |z|^2)
__global__ void __launch_bounds__(kRegThreads) k_reg_phase(float w, float eps2, size_t n, const cf* z, cf* g, double* part) {
  __shared__ double red[kRegThreads / 32];
  double acc[1] = {0.0};
  for (size_t i = (size_t)blockIdx.x * kRegThreads + threadIdx.x; i < n; i += (size_t)kRegBlocks * kRegThreads) {
    const cf v = z[i];
    const float a2 = fmaf(v.x, v.x, v.y * v.y);
    if (a2 == 0.f) continue;
    const float phi = atan2f(v.y, v.x), q = sqrtf(fmaf(phi, phi, eps2));
    acc[0] += (double)(w * q);
    if (g && q > 0.f) { const float c = w * (phi / q) / (2.0f * a2); g[i] = make_float2(fmaf(-c, v.y, g[i].x), fmaf(c, v.x, g[i].y)); }
  }
  block_sum<kRegThreads, 1>(acc, red);
  if (threadIdx.x == 0) part[blockIdx.x] = acc[0];
}

// kind L1 on the Fourier amplitudes of every slice (reading R26c).  The slice has any size, so the transform is the DFT by its
// definition, one axis at a time: one thread per output coefficient, the len twiddles exp(sign 2 pi i m / len) in shared memory (formed
// in double), the index x k mod len advanced by addition, fp64 accumulation.  O(n (nx + ny)) per slice: a regulariser evaluated
// once per iteration on the object (420^2: 0.3 Gflop per slice and pass), not part of the hot path.
constexpr int kDftMaxLen = 4096;
__global__ void __launch_bounds__(256) k_dft_axis(const cf* in, cf* out, int S, int ny, int nx, int axis, double sign, int add) {
  extern __shared__ float2 dft_tw[];
  const int len = axis == 0 ? nx : ny;
  for (int m = threadIdx.x; m < len; m += blockDim.x) {
    double sn, cs_; sincospi(sign * 2.0 * (double)m / (double)len, &sn, &cs_);
    dft_tw[m] = make_float2((float)cs_, (float)sn);
  }
  __syncthreads();
  const size_t os = (size_t)ny * nx, n = (size_t)S * os, i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int s = (int)(i / os), y = (int)((i - (size_t)s * os) / nx), x = (int)(i - (size_t)s * os - (size_t)y * nx);
  const int k = axis == 0 ? x : y;                                    // output index along the axis
  const cf* src = in + (size_t)s * os + (axis == 0 ? (size_t)y * nx : (size_t)x);
  const size_t stride = axis == 0 ? 1 : (size_t)nx;
  double ar = 0.0, ai = 0.0;
  int idx = 0;
  for (int j = 0; j < len; ++j) {
    const cf v = src[(size_t)j * stride]; const float2 w = dft_tw[idx];
    ar += (double)v.x * w.x - (double)v.y * w.y; ai += (double)v.x * w.y + (double)v.y * w.x;
    idx += k; if (idx >= len) idx -= len;
  }
  if (add) out[i] = make_float2((float)((double)out[i].x + ar), (float)((double)out[i].y + ai));
  else out[i] = make_float2((float)ar, (float)ai);
}
// R partials and Z <- dR/dconj(Z) = w Z / (2 sqrt(|Z|^2 + eps^2)) in place
__global__ void __launch_bounds__(kRegThreads) k_reg_fourier_point(float w, float eps2, size_t n, cf* Z, double* part) {
  __shared__ double red[kRegThreads / 32];
  double acc[1] = {0.0};
  for (size_t i = (size_t)blockIdx.x * kRegThreads + threadIdx.x; i < n; i += (size_t)kRegBlocks * kRegThreads) {
    const cf v = Z[i];
    const float r = sqrtf(fmaf(v.x, v.x, fmaf(v.y, v.y, eps2)));
    acc[0] += (double)(w * r);
    const float c = r > 0.f ? 0.5f * w / r : 0.f;
    Z[i] = make_float2(c * v.x, c * v.y);
  }
  block_sum<kRegThreads, 1>(acc, red);
  if (threadIdx.x == 0) part[blockIdx.x] = acc[0];
}

// kinds Tikhonov / TV (in-plane: directions x, y) and their layer versions (direction z): every pixel owns the pair
// (p, p + stride) for the cost and collects, for its gradient, the pair before it and the pair after it
__global__ void __launch_bounds__(kRegThreads) k_reg_diff(int tv, int layer, float w, float eps2, int S, int ny, int nx, const cf* z, cf* g,
                                                        double* part) {
  __shared__ double red[kRegThreads / 32];
  const size_t os = (size_t)ny * nx, n = (size_t)S * os;
  double acc[1] = {0.0};
  for (size_t i = (size_t)blockIdx.x * kRegThreads + threadIdx.x; i < n; i += (size_t)kRegBlocks * kRegThreads) {
    const int s = (int)(i / os), y = (int)((i - (size_t)s * os) / nx), x = (int)(i - (size_t)s * os - (size_t)y * nx);
    const cf c0 = z[i];
    float gx = 0.f, gy = 0.f;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      if (layer ? d != 2 : d == 2) continue;
      const size_t stride = d == 0 ? 1 : d == 1 ? (size_t)nx : os;
      const int c = d == 0 ? x : d == 1 ? y : s, len = d == 0 ? nx : d == 1 ? ny : S;
      if (c + 1 < len) {                                             // pair (i, i + stride): u = z[i + stride] - z[i]
        const cf q = z[i + stride]; const float ux = q.x - c0.x, uy = q.y - c0.y, a2 = fmaf(ux, ux, uy * uy);
        if (!(tv && a2 + eps2 == 0.f)) {
          acc[0] += (double)(w * reg_phi(tv, a2, eps2));
          const float k = w * reg_dphi(tv, a2, eps2); gx -= k * ux; gy -= k * uy;
        }
      }
      if (c > 0) {                                                   // pair (i - stride, i): u = z[i] - z[i - stride]
        const cf q = z[i - stride]; const float ux = c0.x - q.x, uy = c0.y - q.y, a2 = fmaf(ux, ux, uy * uy);
        if (!(tv && a2 + eps2 == 0.f)) { const float k = w * reg_dphi(tv, a2, eps2); gx += k * ux; gy += k * uy; }
      }
    }
    if (g) g[i] = make_float2(g[i].x + gx, g[i].y + gy);
  }
  block_sum<kRegThreads, 1>(acc, red);
  if (threadIdx.x == 0) part[blockIdx.x] = acc[0];
}

__global__ void k_reg_final(const double* part, double* cost) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double s = 0.0;
  for (int b = 0; b < kRegBlocks; ++b) s += part[b];
  *cost += s;
}

// ---- constraints -------------------------------------------------------------------------------------------------
__global__ void k_con_clamp(cf* z, size_t n, float lo, float hi) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const cf v = z[i];
  const float m = sqrtf(fmaf(v.x, v.x, v.y * v.y));
  const float t = m < lo ? lo : (m > hi ? hi : m);
  if (t == m) return;
  z[i] = m > 0.f ? make_float2(v.x * (t / m), v.y * (t / m)) : make_float2(t, 0.f);
}
__global__ void k_con_mask(cf* z, size_t n, size_t os, const float* mask) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float m = mask[i % os];
  z[i] = make_float2(z[i].x * m, z[i].y * m);
}
struct BlurW { int R; float w[65]; };                                 // taps w[t + R], |t| <= R <= 32
__global__ void k_con_blur(const cf* in, cf* out, int S, int ny, int nx, int axis, BlurW bw) {
  const size_t os = (size_t)ny * nx, n = (size_t)S * os, i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int s = (int)(i / os), y = (int)((i - (size_t)s * os) / nx), x = (int)(i - (size_t)s * os - (size_t)y * nx);
  const long stride = axis == 0 ? 1 : axis == 1 ? nx : (long)os;
  const int c = axis == 0 ? x : axis == 1 ? y : s, len = axis == 0 ? nx : axis == 1 ? ny : S;
  float ar = 0.f, ai = 0.f, ws = 0.f;
  for (int t = -bw.R; t <= bw.R; ++t) {
    if (c + t < 0 || c + t >= len) continue;
    const float w = bw.w[t + bw.R]; const cf q = in[(long)i + t * stride];
    ar = fmaf(w, q.x, ar); ai = fmaf(w, q.y, ai); ws += w;
  }
  out[i] = make_float2(ar / ws, ai / ws);
}

// probe support in reciprocal space: z <- Finv(mask .* F(z)); one CTA (CL = 4: one cluster) per mode, the field in
// registers between the two transforms (the chain kernels' FFT)
template <class G>
__global__ void __launch_bounds__(G::T, min_blocks<G>()) k_con_fourier_mask(cf* field, const float* mask) {
  typedef FL<G> F;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int t = threadIdx.x, k = blockIdx.x / G::CL;
  const unsigned rk = Fft<G>::rank();
  ChainSmem<G> cs(smem_raw, t);
  cs.fill_tables(t);
  __syncthreads();
  cf v[32];
  cf* f = field + (size_t)k * F::NNF;
#pragma unroll
  for (int r = 0; r < 32; ++r) v[r] = f[F::pix_y(rk, t, r) * F::NF + F::pix_x(rk, t, r)];
  Fft<G>::fwd(v, cs.sm, cs.tw, cs.tw2, t, rk);
  const float sc = 1.0f / ((float)F::NF * (float)F::NF);
#pragma unroll
  for (int r = 0; r < 32; ++r) v[r] = cscale(v[r], sc * mask[F::fq_y(rk, t, r) * F::NF + F::fq_x(rk, t, r)]);
  Fft<G>::inv(v, cs.sm, cs.tw, cs.tw2, t, rk);
#pragma unroll
  for (int r = 0; r < 32; ++r) f[F::pix_y(rk, t, r) * F::NF + F::pix_x(rk, t, r)] = v[r];
}

// object phase deramp (reading R29), per slice.  Pass 0: block partials of sum z[y+1,x] conj(z[y,x]) and
// sum z[y,x+1] conj(z[y,x]); pass 1 (slopes known): partials of sum z exp(-i(b (y-yc) + c (x-xc))); k_deramp_final sums the
// partials of a slice in fixed order (fp64) and takes the arguments; k_deramp_apply multiplies by the conjugate ramp.
constexpr int kDerampBlocks = 64;                                     // per slice
struct DerampOut { double b, c, a; };
__global__ void __launch_bounds__(256) k_deramp_sums(const cf* z, int ny, int nx, int pass, const DerampOut* slope, double* part /* [S][64][4] */) {
  __shared__ double red[(256 / 32) * 4];
  const int s = blockIdx.y;
  const size_t os = (size_t)ny * nx;
  const cf* zs = z + (size_t)s * os;
  double acc[4] = {0.0, 0.0, 0.0, 0.0};
  const double yc = 0.5 * (ny - 1), xc = 0.5 * (nx - 1);
  const double bb = pass ? slope[s].b : 0.0, cc = pass ? slope[s].c : 0.0;
  for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < os; i += (size_t)kDerampBlocks * 256) {
    const int y = (int)(i / nx), x = (int)(i - (size_t)y * nx);
    const cf c0 = zs[i];
    if (!pass) {
      if (y + 1 < ny) { const cf q = zs[i + nx]; acc[0] += (double)q.x * c0.x + (double)q.y * c0.y; acc[1] += (double)q.y * c0.x - (double)q.x * c0.y; }
      if (x + 1 < nx) { const cf q = zs[i + 1]; acc[2] += (double)q.x * c0.x + (double)q.y * c0.y; acc[3] += (double)q.y * c0.x - (double)q.x * c0.y; }
    } else {
      double sn, cs_; sincos(-(bb * (y - yc) + cc * (x - xc)), &sn, &cs_);
      acc[0] += (double)c0.x * cs_ - (double)c0.y * sn; acc[1] += (double)c0.x * sn + (double)c0.y * cs_;
    }
  }
  block_sum<256, 4>(acc, red);
  if (threadIdx.x == 0)
    for (int c = 0; c < 4; ++c) part[((size_t)s * kDerampBlocks + blockIdx.x) * 4 + c] = acc[c];
}
__global__ void k_deramp_final(const double* part, int pass, DerampOut* out) {
  const int s = blockIdx.x;
  if (threadIdx.x != 0) return;
  double a[4] = {0.0, 0.0, 0.0, 0.0};
  for (int b = 0; b < kDerampBlocks; ++b)
    for (int c = 0; c < 4; ++c) a[c] += part[((size_t)s * kDerampBlocks + b) * 4 + c];
  if (!pass) { out[s].b = atan2(a[1], a[0]); out[s].c = atan2(a[3], a[2]); }
  else out[s].a = atan2(a[1], a[0]);
}
__global__ void k_deramp_apply(cf* z, int ny, int nx, size_t n, const DerampOut* o) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const size_t os = (size_t)ny * nx;
  const int s = (int)(i / os), y = (int)((i - (size_t)s * os) / nx), x = (int)(i - (size_t)s * os - (size_t)y * nx);
  double sn, cs_; sincos(-(o[s].a + o[s].b * (y - 0.5 * (ny - 1)) + o[s].c * (x - 0.5 * (nx - 1))), &sn, &cs_);
  const cf v = z[i];
  z[i] = make_float2((float)((double)v.x * cs_ - (double)v.y * sn), (float)((double)v.x * sn + (double)v.y * cs_));
}

// ---- Adam ----------------------------------------------------------------------------------------------------------
// o1 = 1 - b1, o2 = 1 - b2 formed in double on the host (1 - 0.999f in float is off by 6e-5 relative)
__global__ void k_adam_c(cf* z, const cf* g, cf* m, float* v, size_t n, float lr, float b1, float b2, float o1, float o2, float eps, float ic1, float ic2) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const cf gi = g[i];
  const cf mi = make_float2(fmaf(b1, m[i].x, o1 * gi.x), fmaf(b1, m[i].y, o1 * gi.y));
  const float vi = fmaf(b2, v[i], o2 * fmaf(gi.x, gi.x, gi.y * gi.y));
  m[i] = mi; v[i] = vi;
  const float d = lr * ic1 / (sqrtf(vi * ic2) + eps);
  z[i] = make_float2(fmaf(-d, mi.x, z[i].x), fmaf(-d, mi.y, z[i].y));
}
__global__ void k_adam_r(float* z, const float* g, float* m, float* v, size_t n, float lr, float b1, float b2, float o1, float o2, float eps, float ic1, float ic2) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float mi = fmaf(b1, m[i], o1 * g[i]), vi = fmaf(b2, v[i], o2 * g[i] * g[i]);
  m[i] = mi; v[i] = vi;
  z[i] = fmaf(-lr * ic1 / (sqrtf(vi * ic2) + eps), mi, z[i]);
}

}  // namespace

extern "C" {

size_t ptycho_regularizer_workspace_bytes(void) { return 256 + (size_t)kRegBlocks * sizeof(double); }

int32_t ptycho_cost_regularizer(int32_t kind, float weight, float ref, float eps, int32_t n_slices, int32_t ny, int32_t nx,
                                const pt_c64* field_d, pt_c64* grad_d, double* cost_d, void* workspace_d, size_t workspace_bytes,
                                void* cuda_stream) {
  if (!field_d || !workspace_d) return PT_ERR_NULL;
  if (n_slices < 1 || ny < 1 || nx < 1) return PT_ERR_BAD_SIZE;
  if (kind < PT_REG_L2 || kind > PT_REG_L1_FOURIER || !(eps >= 0.f)) return PT_ERR_BAD_PARAM;
  if (workspace_bytes < ptycho_regularizer_workspace_bytes()) return PT_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  prof_mark(-1, st);
  double* part = (double*)((char*)workspace_d + 256);
  const size_t n = (size_t)n_slices * ny * nx;
  if (kind == PT_REG_L1_FOURIER) {
    if (nx > kDftMaxLen || ny > kDftMaxLen) return PT_ERR_BAD_SIZE;
    if (workspace_bytes < ptycho_regularizer_workspace_bytes() + 2 * n * sizeof(cf)) return PT_ERR_WORKSPACE;
    cf* A = (cf*)((char*)workspace_d + ptycho_regularizer_workspace_bytes());
    cf* B = A + n;
    const unsigned grid = (unsigned)((n + 255) / 256);
    k_dft_axis<<<grid, 256, (size_t)nx * sizeof(float2), st>>>((const cf*)field_d, A, n_slices, ny, nx, 0, -1.0, 0);
    LAUNCH_CHECK(K_regularizer, st);
    k_dft_axis<<<grid, 256, (size_t)ny * sizeof(float2), st>>>(A, B, n_slices, ny, nx, 1, -1.0, 0);
    LAUNCH_CHECK(K_regularizer, st);
    k_reg_fourier_point<<<kRegBlocks, kRegThreads, 0, st>>>(weight, eps * eps, n, B, part);
    LAUNCH_CHECK(K_regularizer, st);
    if (grad_d) {                                                     // F^H: conjugate kernels, columns then rows, added into grad
      k_dft_axis<<<grid, 256, (size_t)ny * sizeof(float2), st>>>(B, A, n_slices, ny, nx, 1, 1.0, 0);
      LAUNCH_CHECK(K_regularizer, st);
      k_dft_axis<<<grid, 256, (size_t)nx * sizeof(float2), st>>>(A, (cf*)grad_d, n_slices, ny, nx, 0, 1.0, 1);
      LAUNCH_CHECK(K_regularizer, st);
    }
  } else if (kind == PT_REG_L1_PHASE)
    k_reg_phase<<<kRegBlocks, kRegThreads, 0, st>>>(weight, eps * eps, n, (const cf*)field_d, (cf*)grad_d, part);
  else if (kind == PT_REG_L2 || kind == PT_REG_L1)
    k_reg_point<<<kRegBlocks, kRegThreads, 0, st>>>(kind == PT_REG_L1, weight, ref, eps * eps, n, (const cf*)field_d, (cf*)grad_d, part);
  else
    k_reg_diff<<<kRegBlocks, kRegThreads, 0, st>>>(kind == PT_REG_TV || kind == PT_REG_LAYER_TV, kind >= PT_REG_LAYER_TIKHONOV, weight,
                                                   eps * eps, n_slices, ny, nx, (const cf*)field_d, (cf*)grad_d, part);
  LAUNCH_CHECK(K_regularizer, st);
  if (cost_d) { k_reg_final<<<1, 32, 0, st>>>(part, cost_d); LAUNCH_CHECK(K_regularizer, st); }
  return PT_OK;
}

int32_t ptycho_apply_constraint(int32_t kind, float a, float b, const float* mask_d, int32_t n_slices, int32_t ny, int32_t nx,
                                pt_c64* field_d, void* workspace_d, size_t workspace_bytes, void* cuda_stream) {
  if (!field_d) return PT_ERR_NULL;
  if (n_slices < 1 || ny < 1 || nx < 1) return PT_ERR_BAD_SIZE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t os = (size_t)ny * nx, n = (size_t)n_slices * os;
  const unsigned grid = (unsigned)((n + 255) / 256);
  prof_mark(-1, st);
  if (kind == PT_CON_AMPLITUDE_CLAMP) {
    if (!(a >= 0.f) || !(b >= a)) return PT_ERR_BAD_PARAM;
    k_con_clamp<<<grid, 256, 0, st>>>((cf*)field_d, n, a, b);
    LAUNCH_CHECK(K_constraint, st);
    return PT_OK;
  }
  if (kind == PT_CON_SUPPORT_MASK) {
    if (!mask_d) return PT_ERR_NULL;
    k_con_mask<<<grid, 256, 0, st>>>((cf*)field_d, n, os, mask_d);
    LAUNCH_CHECK(K_constraint, st);
    return PT_OK;
  }
  if (kind == PT_CON_SUPPORT_MASK_FOURIER) {
    if (!mask_d) return PT_ERR_NULL;
    if (ny != nx || (nx != 64 && nx != 128 && nx != 256)) return PT_ERR_BAD_SIZE;      // the probe sizes of the chain kernels
    cudaError_t e;
    if (nx == 128) {
      if (cudaFuncSetAttribute(k_con_fourier_mask<Geo<128>>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes<Geo<128>>()) != cudaSuccess) return PT_ERR_CUDA;
      e = launch_fft<Geo<128>>(k_con_fourier_mask<Geo<128>>, n_slices * Geo<128>::CL, fft_smem_bytes<Geo<128>>(), st, (cf*)field_d, mask_d);
    } else if (nx == 64) {
      if (cudaFuncSetAttribute(k_con_fourier_mask<Geo<64>>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes<Geo<64>>()) != cudaSuccess) return PT_ERR_CUDA;
      e = launch_fft<Geo<64>>(k_con_fourier_mask<Geo<64>>, n_slices * Geo<64>::CL, fft_smem_bytes<Geo<64>>(), st, (cf*)field_d, mask_d);
    } else {
      if (cudaFuncSetAttribute(k_con_fourier_mask<Geo<256>>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes<Geo<256>>()) != cudaSuccess) return PT_ERR_CUDA;
      e = launch_fft<Geo<256>>(k_con_fourier_mask<Geo<256>>, n_slices * Geo<256>::CL, fft_smem_bytes<Geo<256>>(), st, (cf*)field_d, mask_d);
    }
    if (e != cudaSuccess) return PT_ERR_CUDA;
    LAUNCH_CHECK(K_constraint, st);
    return PT_OK;
  }
  if (kind == PT_CON_PHASE_DERAMP) {
    if (!workspace_d) return PT_ERR_NULL;
    const size_t need = 256 + (size_t)n_slices * (kDerampBlocks * 4 * sizeof(double) + sizeof(DerampOut));
    if (workspace_bytes < need) return PT_ERR_WORKSPACE;
    double* part = (double*)((char*)workspace_d + 256);
    DerampOut* out = (DerampOut*)(part + (size_t)n_slices * kDerampBlocks * 4);
    for (int pass = 0; pass < 2; ++pass) {
      k_deramp_sums<<<dim3(kDerampBlocks, n_slices), 256, 0, st>>>((const cf*)field_d, ny, nx, pass, out, part);
      LAUNCH_CHECK(K_constraint, st);
      k_deramp_final<<<n_slices, 32, 0, st>>>(part, pass, out);
      LAUNCH_CHECK(K_constraint, st);
    }
    k_deramp_apply<<<grid, 256, 0, st>>>((cf*)field_d, ny, nx, n, out);
    LAUNCH_CHECK(K_constraint, st);
    return PT_OK;
  }
  if (kind != PT_CON_LAYER_BLUR && kind != PT_CON_LOWPASS) return PT_ERR_BAD_PARAM;
  if (!(a > 0.f) || a > 8.0f) return PT_ERR_BAD_PARAM;                 // taps |t| <= ceil(4 sigma) <= 32
  if (!workspace_d) return PT_ERR_NULL;
  if (workspace_bytes < n * sizeof(cf)) return PT_ERR_WORKSPACE;
  BlurW bw;
  bw.R = (int)ceil(4.0 * (double)a);
  for (int t = -bw.R; t <= bw.R; ++t) bw.w[t + bw.R] = (float)exp(-(double)t * t / (2.0 * (double)a * (double)a));
  cf* tmp = (cf*)workspace_d;
  if (kind == PT_CON_LAYER_BLUR) {
    k_con_blur<<<grid, 256, 0, st>>>((const cf*)field_d, tmp, n_slices, ny, nx, 2, bw);
    LAUNCH_CHECK(K_constraint, st);
    if (cudaMemcpyAsync(field_d, tmp, n * sizeof(cf), cudaMemcpyDeviceToDevice, st) != cudaSuccess) return PT_ERR_CUDA;
  } else {
    k_con_blur<<<grid, 256, 0, st>>>((const cf*)field_d, tmp, n_slices, ny, nx, 0, bw);
    LAUNCH_CHECK(K_constraint, st);
    k_con_blur<<<grid, 256, 0, st>>>((const cf*)tmp, (cf*)field_d, n_slices, ny, nx, 1, bw);
    LAUNCH_CHECK(K_constraint, st);
  }
  return PT_OK;
}

// ---- ptycho_apply_constraint without a caller's workspace (include/ptycho.h) ----------------------------------------
// The scratch of the blur / low-pass / deramp kernels in a file-scope device array.  In HOST code the name below is a
// host-side stand-in, not a device address (a kernel handed it would fault, or on a GPU that can reach host memory use the
// wrong memory): the address comes from cudaGetSymbolAddress, once per device with that device current, and is cached.
// Every call on a device shares the array; nothing in it has to start at zero (see the header).
static __device__ __align__(256) unsigned char g_static_scratch[PT_STATIC_SCRATCH_BYTES];
constexpr int kStaticMaxDevices = 64;
static std::atomic<void*> g_static_scratch_ptr[kStaticMaxDevices];

int32_t ptycho_apply_constraint_static(int32_t kind, float a, int32_t n_slices, int32_t ny, int32_t nx, pt_c64* field_d,
                                       void* cuda_stream) {
  if (!field_d) return PT_ERR_NULL;
  if (n_slices < 1 || ny < 1 || nx < 1) return PT_ERR_BAD_SIZE;
  size_t need;
  if (kind == PT_CON_LAYER_BLUR || kind == PT_CON_LOWPASS) need = (size_t)n_slices * ny * nx * sizeof(cf);
  else if (kind == PT_CON_PHASE_DERAMP) need = 256 + (size_t)n_slices * (kDerampBlocks * 4 * sizeof(double) + sizeof(DerampOut));
  else return kind >= PT_CON_AMPLITUDE_CLAMP && kind <= PT_CON_PHASE_DERAMP ? PT_ERR_UNSUPPORTED : PT_ERR_BAD_PARAM;
  if (need > (size_t)PT_STATIC_SCRATCH_BYTES) return PT_ERR_STATIC_LIMIT;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kStaticMaxDevices) return PT_ERR_CUDA;
  void* scratch = g_static_scratch_ptr[dev].load(std::memory_order_acquire);
  if (!scratch) {                                                      // set-up, once per device (threads racing here store the same value)
    if (cudaGetSymbolAddress(&scratch, g_static_scratch) != cudaSuccess || !scratch) return PT_ERR_CUDA;
    g_static_scratch_ptr[dev].store(scratch, std::memory_order_release);
  }
  return ptycho_apply_constraint(kind, a, 0.f, nullptr, n_slices, ny, nx, field_d, scratch, (size_t)PT_STATIC_SCRATCH_BYTES, cuda_stream);
}

static int adam_params(const void* z, const void* g, const void* m, const void* v, float b1, float b2, float eps, int32_t step,
                       float* ic1, float* ic2) {
  if (!z || !g || !m || !v) return PT_ERR_NULL;
  if (step < 1 || !(b1 >= 0.f && b1 < 1.f) || !(b2 >= 0.f && b2 < 1.f) || !(eps >= 0.f)) return PT_ERR_BAD_PARAM;
  *ic1 = (float)(1.0 / (1.0 - pow((double)b1, (double)step)));
  *ic2 = (float)(1.0 / (1.0 - pow((double)b2, (double)step)));
  return PT_OK;
}

int32_t ptycho_adam_update(pt_c64* z_d, const pt_c64* g_d, pt_c64* m_d, float* v_d, size_t n, float lr, float beta1, float beta2,
                           float eps, int32_t step, void* cuda_stream) {
  float ic1, ic2;
  int rc = adam_params(z_d, g_d, m_d, v_d, beta1, beta2, eps, step, &ic1, &ic2);
  if (rc != PT_OK) return rc;
  if (n == 0) return PT_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  prof_mark(-1, st);
  k_adam_c<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((cf*)z_d, (const cf*)g_d, (cf*)m_d, v_d, n, lr, beta1, beta2, (float)(1.0 - (double)beta1), (float)(1.0 - (double)beta2), eps, ic1, ic2);
  LAUNCH_CHECK(K_adam, st);
  return PT_OK;
}

int32_t ptycho_adam_update_real(float* z_d, const float* g_d, float* m_d, float* v_d, size_t n, float lr, float beta1, float beta2,
                                float eps, int32_t step, void* cuda_stream) {
  float ic1, ic2;
  int rc = adam_params(z_d, g_d, m_d, v_d, beta1, beta2, eps, step, &ic1, &ic2);
  if (rc != PT_OK) return rc;
  if (n == 0) return PT_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  prof_mark(-1, st);
  k_adam_r<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(z_d, g_d, m_d, v_d, n, lr, beta1, beta2, (float)(1.0 - (double)beta1), (float)(1.0 - (double)beta2), eps, ic1, ic2);
  LAUNCH_CHECK(K_adam, st);
  return PT_OK;
}

}  // extern "C"
