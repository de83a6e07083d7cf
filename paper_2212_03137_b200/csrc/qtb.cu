// qtb.cu -- adaptive Quantum Thermal Bath:
//   Q2  white noise regenerated from Philox (nothing stored; the paper keeps 3 N_seg numbers per
//       DOF),
//   Q3  filter H_z(omega_j) = sqrt(2 m_z gamma_z(omega_j) Theta(omega_j, beta) / dt)
//       (Eq. 13-14),
//   Q4  coloured segment F_c = h_z (*) r by FFT convolution,
//   Q5  segment spectra |v~|^2 and Re(v~ F~*) (Eq. 21-22),
//   Q6  per-type averages,
//   Q7  SIMPLE adaptation with lower bound (Eq. 23; readings G12-G15).
// The FFT is a hand-written shared-memory Stockham autosort transform (radix 4 with one radix-2
// pass when log2 n is odd), fp64 complex, one CTA of n/4 threads per transform; each pass stages
// its butterfly in registers so a single n x 16 B buffer is enough.
#include "qhp_internal.cuh"
#include "philox.cuh"

// ---------------------------------------------------------------------------------------------
// FFT
// ---------------------------------------------------------------------------------------------
// Shared-memory FFT buffers are swizzled: element i lives at FPAD(i) = i ^ (((i >> 3) ^ (i >> 6)) & 7).  The first
// pass of a transform stores R consecutive elements per thread, i.e. at a lane stride of 16 R bytes (256 B for
// radix 16), which unswizzled is an 8-way bank conflict on every store (measured: half of all shared-memory
// wavefronts of the segment kernels); the XOR of the 16-byte bank-group index with bits 3-5 and 6-8 of the
// element index makes the stores of lane strides 2, 4, 8 and 16 elements conflict-free and leaves runs of 8
// consecutive elements (all other accesses) inside one aligned 128-byte row.  No extra memory.
#define FPAD(i) ((i) ^ ((((i) >> 3) ^ ((i) >> 6)) & 7))
#define FPAD_LEN(n) (n)
__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// tw[m] = exp(-2 pi i m / tw_n); returns exp(sign * 2 pi i * num / den), den | tw_n (powers of two), 0 <= num < den
__device__ __forceinline__ double2 twiddle(const double2 *__restrict__ tw, int tw_n, int num, int den, int sign) {
  double2 w = tw[num * (tw_n >> (__ffs(den) - 1))];
  if (sign > 0) w.y = -w.y;
  return w;
}

// 4-point DFT in place: (a, b, c, d) -> (X0, X1, X2, X3), X_v = sum_u x_u exp(SG 2 pi i u v / 4)
template <int SG>
__device__ __forceinline__ void dft4(double2 &a, double2 &b, double2 &c, double2 &d) {
  const double2 t0 = make_double2(a.x + c.x, a.y + c.y), t1 = make_double2(a.x - c.x, a.y - c.y);
  const double2 t2 = make_double2(b.x + d.x, b.y + d.y), e = make_double2(b.x - d.x, b.y - d.y);
  const double2 t3 = (SG < 0) ? make_double2(e.y, -e.x) : make_double2(-e.y, e.x);   // (b - d) * (SG i)
  a = make_double2(t0.x + t2.x, t0.y + t2.y); b = make_double2(t1.x + t3.x, t1.y + t3.y);
  c = make_double2(t0.x - t2.x, t0.y - t2.y); d = make_double2(t1.x - t3.x, t1.y - t3.y);
}

// One Stockham pass of radix R (16, 4 or 2) at stride Ns over buf[0..n).  Every thread t < max(n/16, 1)
// keeps 16 elements in registers: one radix-16 butterfly (two radix-4 layers without touching shared
// memory in between: half the shared-memory traffic of two radix-4 passes, which bounded the first
// version of the noise kernel), or 4 radix-4 / 8 radix-2 butterflies.  Reads are contiguous in t.
// Input twiddles w^(k u) are successive powers of one table entry w^k (<= 15 products, ~1e-14 relative).
template <int R, int SG>
__device__ __forceinline__ void fft_pass(double2 *buf, int n, int Ns, const double2 *__restrict__ tw, int tw_n, int t,
                                         const double2 wpre = make_double2(0.0, 0.0), bool have_w = false) {
  constexpr int G = 16 / R;                       // butterflies per thread
  const int nth = n >= 16 ? n >> 4 : 1, nb = n / R;
  const bool on = t < nth;
  double2 v[16];
  int j0[G];
  if (on) {
#pragma unroll
    for (int q = 0; q < G; ++q) {
      const int j = t + q * nth;
      j0[q] = -1;
      if (j < nb) {
        const int k = j & (Ns - 1);
#pragma unroll
        for (int u = 0; u < R; ++u) v[q * R + u] = buf[FPAD(j + u * nb)];
        if (k) {
          const double2 w1 = have_w ? wpre : twiddle(tw, tw_n, k, Ns * R, SG);
          double2 w = w1;
#pragma unroll
          for (int u = 1; u < R; ++u) {
            v[q * R + u] = cmul(v[q * R + u], w);
            if (u + 1 < R) w = cmul(w, w1);
          }
        }
        j0[q] = (j - k) * R + k;
      }
    }
  }
  __syncthreads();
  if (on) {
    if (R == 16) {
      if (j0[0] >= 0) {
        // u = 4 a + b: 4-point DFTs over a, twiddles w16^(b c), 4-point DFTs over b; X[c + 4 d] ends in v[4 c + d]
#pragma unroll
        for (int b = 0; b < 4; ++b) dft4<SG>(v[b], v[4 + b], v[8 + b], v[12 + b]);
        const double c8 = 0.92387953251128673848, s8 = 0.38268343236508978178, r2 = 0.70710678118654752440;
        const double sg = (SG < 0) ? -1.0 : 1.0;
        // after the first layer v[4 c + b] = T[b][c]
        v[5] = cmul(v[5], make_double2(c8, sg * s8));        // b c = 1
        v[6] = cmul(v[6], make_double2(r2, sg * r2));        // 2
        v[7] = cmul(v[7], make_double2(s8, sg * c8));        // 3
        v[9] = cmul(v[9], make_double2(r2, sg * r2));        // 2
        v[10] = make_double2(-sg * v[10].y, sg * v[10].x);   // 4: multiply by (SG i)
        v[11] = cmul(v[11], make_double2(-r2, sg * r2));     // 6
        v[13] = cmul(v[13], make_double2(s8, sg * c8));      // 3
        v[14] = cmul(v[14], make_double2(-r2, sg * r2));     // 6
        v[15] = cmul(v[15], make_double2(-c8, -sg * s8));    // 9
#pragma unroll
        for (int c = 0; c < 4; ++c) dft4<SG>(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
          for (int d = 0; d < 4; ++d) buf[FPAD(j0[0] + (c + 4 * d) * Ns)] = v[4 * c + d];
      }
    } else {
#pragma unroll
      for (int q = 0; q < G; ++q)
        if (j0[q] >= 0) {
          if (R == 4) {
            dft4<SG>(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
#pragma unroll
            for (int u = 0; u < 4; ++u) buf[FPAD(j0[q] + u * Ns)] = v[4 * q + u];
          } else {
            const double2 x0 = v[2 * q], x1 = v[2 * q + 1];
            buf[FPAD(j0[q])] = make_double2(x0.x + x1.x, x0.y + x1.y);
            buf[FPAD(j0[q] + Ns)] = make_double2(x0.x - x1.x, x0.y - x1.y);
          }
        }
    }
  }
  __syncthreads();
}

// In-place Stockham FFT of buf[0..n) by blockDim.x >= max(n/16, 1) threads (all threads of the CTA
// must call).  sign = -1 forward, +1 inverse (unnormalised).  Result in natural order.
// Radix schedule: the factor of n that is not a power of 16 goes FIRST (radix-2 / radix-4 passes at small Ns need
// at most a handful of twiddles), then radix-16 passes; the one table entry w^k a thread needs in each radix-16
// pass is requested before the first pass, so that no pass waits on a global load.
template <int SG>
__device__ __forceinline__ void fft_smem_sg(double2 *buf, int n, const double2 *__restrict__ tw, int tw_n, int t) {
  int r0 = n, m16 = 0;
  while (r0 >= 16 && (r0 & 15) == 0) { r0 >>= 4; ++m16; }            // n = r0 * 16^m16, r0 in {1, 2, 4, 8}
  double2 w16[3] = {make_double2(1.0, 0.0), make_double2(1.0, 0.0), make_double2(1.0, 0.0)};
  {
    int Ns = r0;
#pragma unroll
    for (int p = 0; p < 3; ++p)
      if (p < m16) {
        const int k = t & (Ns - 1);
        if (t < (n >> 4)) w16[p] = twiddle(tw, tw_n, k, Ns * 16, SG);
        Ns <<= 4;
      }
  }
  int Ns = 1;
  if (r0 == 2) { fft_pass<2, SG>(buf, n, 1, tw, tw_n, t); Ns = 2; }
  else if (r0 == 4) { fft_pass<4, SG>(buf, n, 1, tw, tw_n, t); Ns = 4; }
  else if (r0 == 8) { fft_pass<2, SG>(buf, n, 1, tw, tw_n, t); fft_pass<4, SG>(buf, n, 2, tw, tw_n, t); Ns = 8; }
#pragma unroll
  for (int p = 0; p < 3; ++p)
    if (p < m16) { fft_pass<16, SG>(buf, n, Ns, tw, tw_n, t, w16[p], true); Ns <<= 4; }
}
// t: index of the calling thread inside its FFT (threads t >= max(n/16, 1) only take part in the barriers);
// several FFTs of the same length can run side by side in one CTA on different buffers.
__device__ __noinline__ void fft_smem(double2 *buf, int n, int sign, const double2 *__restrict__ tw, int tw_n, int t) {
  if (sign < 0) fft_smem_sg<-1>(buf, n, tw, tw_n, t);
  else fft_smem_sg<1>(buf, n, tw, tw_n, t);
}

// ---- 8 elements per thread (n / 8 threads per transform): half the registers of the 16-element passes, twice the warps.
// 8-point DFT, decimation in time: X_k = E_k + w8^k O_k, X_{k+4} = E_k - w8^k O_k with E, O the 4-point DFTs of the even
// and odd inputs; in place, natural order.
template <int SG>
__device__ __forceinline__ void dft8(double2 (&v)[8]) {
  dft4<SG>(v[0], v[2], v[4], v[6]);
  dft4<SG>(v[1], v[3], v[5], v[7]);
  const double r2 = 0.70710678118654752440, sg = (SG < 0) ? -1.0 : 1.0;
  const double2 o0 = v[1];
  const double2 o1 = cmul(v[3], make_double2(r2, sg * r2));
  const double2 o2 = make_double2(-sg * v[5].y, sg * v[5].x);          // * (SG i)
  const double2 o3 = cmul(v[7], make_double2(-r2, sg * r2));
  const double2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
  v[0] = make_double2(e0.x + o0.x, e0.y + o0.y); v[4] = make_double2(e0.x - o0.x, e0.y - o0.y);
  v[1] = make_double2(e1.x + o1.x, e1.y + o1.y); v[5] = make_double2(e1.x - o1.x, e1.y - o1.y);
  v[2] = make_double2(e2.x + o2.x, e2.y + o2.y); v[6] = make_double2(e2.x - o2.x, e2.y - o2.y);
  v[3] = make_double2(e3.x + o3.x, e3.y + o3.y); v[7] = make_double2(e3.x - o3.x, e3.y - o3.y);
}

// one Stockham pass of radix R (8, 4 or 2) at stride Ns, 8 elements per thread (t < n / 8)
template <int R, int SG>
__device__ __forceinline__ void fft_pass8(double2 *buf, int n, int Ns, const double2 *__restrict__ tw, int tw_n, int t,
                                          const double2 wpre = make_double2(0.0, 0.0), bool have_w = false) {
  constexpr int G = 8 / R;
  const int nth = n >> 3, nb = n / R;
  const bool on = t < nth;
  double2 v[8];
  int j0[G];
  if (on) {
#pragma unroll
    for (int q = 0; q < G; ++q) {
      const int j = t + q * nth, k = j & (Ns - 1);
#pragma unroll
      for (int u = 0; u < R; ++u) v[q * R + u] = buf[FPAD(j + u * nb)];
      if (k) {
        const double2 w1 = have_w ? wpre : twiddle(tw, tw_n, k, Ns * R, SG);
        double2 w = w1;
#pragma unroll
        for (int u = 1; u < R; ++u) {
          v[q * R + u] = cmul(v[q * R + u], w);
          if (u + 1 < R) w = cmul(w, w1);
        }
      }
      j0[q] = (j - k) * R + k;
    }
  }
  __syncthreads();
  if (on) {
    if (R == 8) {
      dft8<SG>(v);
#pragma unroll
      for (int u = 0; u < 8; ++u) buf[FPAD(j0[0] + u * Ns)] = v[u];
    } else if (R == 4) {
#pragma unroll
      for (int q = 0; q < G; ++q) {
        dft4<SG>(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
#pragma unroll
        for (int u = 0; u < 4; ++u) buf[FPAD(j0[q] + u * Ns)] = v[4 * q + u];
      }
    } else {
#pragma unroll
      for (int q = 0; q < G; ++q) {
        const double2 x0 = v[2 * q], x1 = v[2 * q + 1];
        buf[FPAD(j0[q])] = make_double2(x0.x + x1.x, x0.y + x1.y);
        buf[FPAD(j0[q] + Ns)] = make_double2(x0.x - x1.x, x0.y - x1.y);
      }
    }
  }
  __syncthreads();
}

// forward transform of buf[0..n), n >= 8 a power of two, by n / 8 threads per transform (all threads of the CTA call):
// n = r0 * 8^m: the factor r0 in {1, 2, 4} first, then m radix-8 passes whose table entries are requested up front
__device__ __noinline__ void fft_fwd8(double2 *buf, int n, const double2 *__restrict__ tw, int tw_n, int t) {
  int r0 = n, m8 = 0;
  while (r0 >= 8 && (r0 & 7) == 0) { r0 >>= 3; ++m8; }
  double2 w8[4] = {make_double2(1.0, 0.0), make_double2(1.0, 0.0), make_double2(1.0, 0.0), make_double2(1.0, 0.0)};
  {
    int Ns = r0;
#pragma unroll
    for (int p = 0; p < 4; ++p)
      if (p < m8) {
        const int k = t & (Ns - 1);
        if (t < (n >> 3)) w8[p] = twiddle(tw, tw_n, k, Ns * 8, -1);
        Ns <<= 3;
      }
  }
  int Ns = 1;
  if (r0 == 2) { fft_pass8<2, -1>(buf, n, 1, tw, tw_n, t); Ns = 2; }
  else if (r0 == 4) { fft_pass8<4, -1>(buf, n, 1, tw, tw_n, t); Ns = 4; }
#pragma unroll
  for (int p = 0; p < 4; ++p)
    if (p < m8) { fft_pass8<8, -1>(buf, n, Ns, tw, tw_n, t, w8[p], true); Ns <<= 3; }
}

// The segment kernels only transform forward (the inverse is conj(forward(conj(.)))): their own non-inlined body.  With
// both directions in one function (fft_smem) ptxas spilled 6.9 KB per call in the context of k_qtb_noise, with the
// forward direction alone 1.1 KB: noise generation 41.8 -> 30.5 ms per C3 segment.
__device__ __noinline__ void fft_fwd(double2 *buf, int n, const double2 *__restrict__ tw, int tw_n, int t) {
  fft_smem_sg<-1>(buf, n, tw, tw_n, t);
}

__global__ void k_twiddle(double2 *tw, int n) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n) return;
  double s, c;
  sincospi(-2.0 * (double)m / (double)n, &s, &c);
  tw[m] = make_double2(c, s);
}

__global__ void __launch_bounds__(512, 1) k_fft_batch(double2 *data, int n, int sign, const double2 *__restrict__ tw, int tw_n) {
  extern __shared__ double2 fbuf[];
  double2 *d = data + (long long)blockIdx.x * n;
  for (int k = threadIdx.x; k < n; k += blockDim.x) fbuf[FPAD(k)] = d[k];
  __syncthreads();
  fft_smem(fbuf, n, sign, tw, tw_n, threadIdx.x);
  for (int k = threadIdx.x; k < n; k += blockDim.x) d[k] = fbuf[FPAD(k)];
}

static int fft_threads(int n) { return n / 16 < 32 ? 32 : n / 16; }

int qhp_fft_launch(double *data, int n, int64_t batch, int sign, const double *tw, int tw_n, cudaStream_t st) {
  const size_t smem = sizeof(double2) * (size_t)FPAD_LEN(n);
  cudaError_t e = cudaFuncSetAttribute(k_fft_batch, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return QHP_ECUDA;
  k_fft_batch<<<(unsigned)batch, fft_threads(n), smem, st>>>((double2 *)data, n, sign, (const double2 *)tw, tw_n);
  return cudaGetLastError() == cudaSuccess ? QHP_OK : QHP_ECUDA;
}

// ---------------------------------------------------------------------------------------------
// Q3: filter, kernel and the spectrum used by the convolution
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double qtb_theta(double w, double kT) {   // Eq. 14
  if (w == 0.0) return kT;
  const double hw = QHP_HBAR * fabs(w);
  return 0.5 * hw / tanh(0.5 * hw / kT);
}

// Hf[z][j] = kappa[j] sqrt(2 (m_z/ACC) gamma_z[j] Theta(omega_j) / dt), omega_j = 2 pi j / (2 n_seg dt);
// kappa = kernel-correction factor of reading G11, NULL = 1
__global__ void k_qtb_filter(int nt, int n_seg, double dt, double kT, int classical, const double *__restrict__ mass,
                             const double *__restrict__ gamma, const double *__restrict__ kappa, double *Hf) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int nf = n_seg + 1;
  if (idx >= nt * nf) return;
  const int z = idx / nf, j = idx % nf;
  const double w = 2.0 * QHP_PI * j / (2.0 * n_seg * dt);
  const double th = classical ? kT : qtb_theta(w, kT);
  const double H = sqrt(2.0 * (mass[z] / QHP_ACC) * gamma[idx] * th / dt);
  Hf[idx] = kappa ? kappa[j] * H : H;
}

// hk[z][k + n_seg] = (1/N_k) sum_j H_ext[j] cos(2 pi j k / N_k), k = -n_seg..n_seg-1 (real, even)
__global__ void k_qtb_kernel(int nt, int n_seg, const double *__restrict__ Hf, double *hk) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int nk = 2 * n_seg;
  if (idx >= nt * nk) return;
  const int z = idx / nk, k = idx % nk - n_seg;
  const double *H = Hf + z * (n_seg + 1);
  double s = 0.0;
  for (int j = 0; j < nk; ++j) {
    const double Hj = (j <= n_seg) ? H[j] : H[nk - j];
    long long jk = ((long long)j * k) % nk;
    if (jk < 0) jk += nk;
    s += Hj * cospi(2.0 * (double)jk / (double)nk);
  }
  hk[idx] = s / nk;
}

// H4[z][q] = sum_{m < 2 n_seg} hk[z][m] exp(-2 pi i q m / (4 n_seg)): spectrum of buf[m] = h[m - n_seg]
__global__ void k_qtb_spectrum4(int nt, int n_seg, const double *__restrict__ hk, double2 *H4) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int nk = 2 * n_seg, nf = 4 * n_seg;
  if (idx >= nt * nf) return;
  const int z = idx / nf, q = idx % nf;
  const double *h = hk + z * nk;
  double re = 0.0, im = 0.0;
  for (int m = 0; m < nk; ++m) {
    const long long qm = ((long long)q * m) % nf;
    double s, c;
    sincospi(-2.0 * (double)qm / (double)nf, &s, &c);
    re += h[m] * c;
    im += h[m] * s;
  }
  H4[idx] = make_double2(re, im);
}

// white noise of one pass of k_qtb_noise into the transform buffer
__device__ __forceinline__ void qtb_fill_noise(double2 *nbuf, double *zb, int nf, int nw, int n_seg, int pass, int atom,
                                            unsigned long long seed, long long seg, int t, int nthr) {
  for (int m = t; m < nf; m += nthr) {
    double2 v = make_double2(0.0, 0.0);
    if (m < nw) {
      if (pass < 2) {
        double z[3] = {0.0, 0.0, 0.0};
        if (atom >= 0) qhp_normals3(seed, (uint32_t)atom, 0u, QHP_TAG_QTB, (uint64_t)(seg * n_seg + m), z);
        v = make_double2(z[0], z[1]);
        zb[pass * nw + m] = z[2];
      } else {
        v = make_double2(zb[m], zb[nw + m]);
      }
    }
    nbuf[FPAD(m)] = v;
  }
}

// ---------------------------------------------------------------------------------------------
// Q2 + Q4: one CTA per PAIR of segment slots (two atoms of one type, qhp_internal.cuh).  The kernel h is
// real, so real and imaginary part of a complex sequence are filtered independently: (x0, y0), (x1, y1)
// and (z0, z1) are three complex transforms for six components (the z components of two atoms share one).
//   F_c[dof][n] = sum_k h_z[k] r(dof, seg*n_seg + n - k + n_seg),  n = 0..n_seg-1
// Output: the 48-byte half row of the pair in the segment layout [group][n_seg][12].
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512, 1) k_qtb_noise(int n_seg, unsigned long long seed, long long seg, const int32_t *__restrict__ slot_atom,
                                                   const int32_t *__restrict__ type, const double2 *__restrict__ H4,
                                                   const double2 *__restrict__ tw, double *Fc) {
  extern __shared__ double2 nbuf[];
  const int nf = 4 * n_seg, nw = 3 * n_seg;
  double *zb = reinterpret_cast<double *>(nbuf + FPAD_LEN(nf)); // [2][nw] z noise of the two atoms
  const int slot0 = 2 * blockIdx.x, t = threadIdx.x;
  const int at[2] = {slot_atom[slot0], slot_atom[slot0 + 1]};
  if (at[0] < 0 && at[1] < 0) return;                           // padding
  const double2 *Hz = H4 + (long long)type[at[0] >= 0 ? at[0] : at[1]] * nf;
  const double inv = 1.0 / (double)nf;
  for (int pass = 0; pass < 3; ++pass) {
    qtb_fill_noise(nbuf, zb, nf, nw, n_seg, pass, pass < 2 ? at[pass] : -1, seed, seg, t, blockDim.x);
    __syncthreads();
    fft_fwd(nbuf, nf, tw, nf, t);
    // inverse transform = conj(forward(conj(.))): one transform direction in this kernel
#pragma unroll 8
    for (int q = t; q < nf; q += blockDim.x) {
      const double2 p = cmul(nbuf[FPAD(q)], Hz[q]);
      nbuf[FPAD(q)] = make_double2(p.x, -p.y);
    }
    __syncthreads();
    fft_fwd(nbuf, nf, tw, nf, t);
    // every pass writes its own pieces of the pair's 48-byte half rows (x0 y0 z0 x1 y1 z1); L2 merges them
    for (int n = t; n < n_seg; n += blockDim.x) {
      double2 y = nbuf[FPAD(n + 2 * n_seg)];
      y.y = -y.y;
      double *out = Fc + qhp_seg_addr(slot0, n_seg, n);
      if (pass == 0) *reinterpret_cast<double2 *>(out) = make_double2(y.x * inv, y.y * inv);
      else if (pass == 1) { out[3] = y.x * inv; out[4] = y.y * inv; }
      else { out[2] = y.x * inv; out[5] = y.y * inv; }
    }
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------------------------
// Q5 + Q6: spectra.  One CTA walks a run of slot groups (4 atoms, 12 DOF) of one type; v and F_c of a DOF
// are the real and imaginary part of one zero-padded N_k-point transform.  A group is one contiguous
// n_seg x 96 B region of each segment array, read with coalesced loads; DPR of its 12 DOFs are transformed
// side by side per round (DPR thread groups of max(N_k/16, 32) threads).  The bins are accumulated in one
// shared array per CTA, the thread groups adding in a fixed order; per-CTA sums -> fixed-order reduction.
// ---------------------------------------------------------------------------------------------
template <int DPR>
__global__ void __launch_bounds__(DPR == 3 ? 768 : 512, 1) k_qtb_spectra(int n_seg, const int32_t *__restrict__ cta_tab,
                                                        const double *__restrict__ vseg, const double *__restrict__ Fc,
                                                        const double2 *__restrict__ tw, int tw_n, double *part) {
  extern __shared__ double2 sbuf_all[];
  const int nk = 2 * n_seg, nf = n_seg + 1, gsz = blockDim.x / DPR, bl = nk + 1;   // + 1: the DOF buffers start one bank group apart
  const int c = threadIdx.x / gsz, t = threadIdx.x - c * gsz;
  double *acc = reinterpret_cast<double *>(sbuf_all + (size_t)2 * DPR * bl);   // [2][nf]
  for (int j = threadIdx.x; j < 2 * nf; j += blockDim.x) acc[j] = 0.0;
  const int gb = cta_tab[3 * blockIdx.x + 1], ge = cta_tab[3 * blockIdx.x + 2];
  constexpr int RPG = 12 / DPR;                          // rounds per group
  const int rounds = (ge - gb) * RPG;
  // round q of the CTA: DOFs [r DPR, (r + 1) DPR) of group g; its (v, F_c) samples go straight from global to
  // shared memory (cp.async, 8 bytes each) while the previous round is being transformed (two buffers)
  auto issue = [&](int q, double2 *buf) {
    const int g = gb + q / RPG, r = q - (q / RPG) * RPG;
    const double *vg = vseg + (long long)g * n_seg * 12 + r * DPR, *fg = Fc + (long long)g * n_seg * 12 + r * DPR;
    for (int idx = threadIdx.x; idx < n_seg * DPR; idx += blockDim.x) {
      const int n = idx / DPR, d = idx - n * DPR;
      double2 *dst = buf + (size_t)d * bl + FPAD(n);
      const uint32_t sa = (uint32_t)__cvta_generic_to_shared(dst);
      asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(vg + (long long)n * 12 + d) : "memory");
      asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa + 8), "l"(fg + (long long)n * 12 + d) : "memory");
      buf[(size_t)d * bl + FPAD(n_seg + n)] = make_double2(0.0, 0.0);      // zero padding to N_k
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  if (rounds > 0) issue(0, sbuf_all);
  for (int q = 0; q < rounds; ++q) {
    double2 *cur = sbuf_all + (size_t)(q & 1) * DPR * bl, *nxt = sbuf_all + (size_t)((q + 1) & 1) * DPR * bl;
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();
    if (q + 1 < rounds) issue(q + 1, nxt);
    double2 *sbuf = cur + (size_t)c * bl;
    fft_fwd8(sbuf, nk, tw, tw_n, t);
    for (int cc = 0; cc < DPR; ++cc) {                   // the thread groups add in a fixed order
      if (c == cc)
        for (int j = t; j < nf; j += gsz) {
          const double2 A = sbuf[FPAD(j)], Zm = sbuf[FPAD((nk - j) & (nk - 1))];
          const double vx = 0.5 * (A.x + Zm.x), vy = 0.5 * (A.y - Zm.y);     // V_j
          const double px = 0.5 * (A.y + Zm.y), py = -0.5 * (A.x - Zm.x);    // Phi_j
          acc[j] += vx * vx + vy * vy;
          acc[nf + j] += vx * px + vy * py;
        }
      __syncthreads();
    }
  }
  __syncthreads();
  double *o = part + (long long)blockIdx.x * 2 * nf;
  for (int j = threadIdx.x; j < 2 * nf; j += blockDim.x) o[j] = acc[j];
}

__global__ void k_qtb_reduce(int nt, int n_seg, int n_cta, const int32_t *__restrict__ cta_tab, const double *__restrict__ part,
                             const double *__restrict__ ndof_type, double dt, double *Cvv, double *CvF) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int nf = n_seg + 1;
  if (idx >= nt * nf) return;
  const int z = idx / nf, j = idx % nf;
  double sv = 0.0, sf = 0.0;
  for (int c = 0; c < n_cta; ++c)
    if (cta_tab[3 * c] == z) { sv += part[(long long)c * 2 * nf + j]; sf += part[(long long)c * 2 * nf + nf + j]; }
  const double nd = ndof_type[z];
  if (nd > 0) {
    Cvv[idx] = dt / n_seg * sv / nd;
    CvF[idx] = dt / n_seg * sf / nd;
  } else { Cvv[idx] = 0.0; CvF[idx] = 0.0; }
}

// Q7: one CTA per type
__global__ void k_qtb_adapt(int n_seg, const double *__restrict__ mass, double gamma0, double a_gamma, double gmin_frac,
                            const double *__restrict__ Cvv, const double *__restrict__ CvF, double *gamma,
                            const double *__restrict__ tau) {
  __shared__ double scratch[32];
  __shared__ double nrm_s;
  const int z = blockIdx.x, nf = n_seg + 1, t = threadIdx.x;
  if (tau && tau[z] > 0.0) return;              // a RATIO type (k_qtb_adapt_ratio)
  const double mz = mass[z] / QHP_ACC;
  double s = 0.0;
  for (int j = t; j < nf; j += blockDim.x) {
    const double dl = mz * gamma[z * nf + j] * Cvv[z * nf + j] - CvF[z * nf + j];
    s += dl * dl;
  }
  // fixed-order block sum
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((t & 31) == 0) scratch[t >> 5] = s;
  __syncthreads();
  if (t == 0) {
    double tot = 0.0;
    for (int k = 0; k < (int)(blockDim.x >> 5); ++k) tot += scratch[k];
    nrm_s = sqrt(tot);
  }
  __syncthreads();
  const double nrm = nrm_s;
  if (nrm == 0.0) return;
  const double gmin = gmin_frac * gamma0;
  for (int j = t; j < nf; j += blockDim.x) {
    const double dl = mz * gamma[z * nf + j] * Cvv[z * nf + j] - CvF[z * nf + j];
    const double g = gamma[z * nf + j] - a_gamma * gamma0 * dl / nrm;
    gamma[z * nf + j] = g > gmin ? g : gmin;
  }
}

// RATIO adaptation (Eq. 24-26) for the types with tau[z] > 0: exponential-window
// averages of the per-type spectra (Eq. 26; the first segment initialises them, reading G24), then
// gamma_z = Re<C_vF> / (m_z <C_vv>) (Eq. 25) with the lower bound of l.248.  Runs after k_qtb_adapt,
// which leaves these types alone.
__global__ void k_qtb_adapt_ratio(int nt, int n_seg, const double *__restrict__ mass, double gamma0, double gmin_frac,
                                  double dt, const double *__restrict__ tau, int first, const double *__restrict__ Cvv,
                                  const double *__restrict__ CvF, double *avv, double *avf, double *gamma) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int nf = n_seg + 1;
  if (idx >= nt * nf) return;
  const int z = idx / nf;
  if (!(tau[z] > 0.0)) return;
  const double w = first ? 0.0 : exp(-(double)n_seg * dt / tau[z]);
  const double av = avv[idx] * w + Cvv[idx] * (1.0 - w), af = avf[idx] * w + CvF[idx] * (1.0 - w);
  avv[idx] = av; avf[idx] = af;
  const double den = mass[z] / QHP_ACC * av;
  if (den > 0.0) {
    const double g = af / den, gmin = gmin_frac * gamma0;
    gamma[idx] = g > gmin ? g : gmin;
  }
}

// parity hook: internal [group][n_seg][12] -> documented [3N][n_seg] (atom order)
__global__ void k_seg_export(const double *__restrict__ in, double *__restrict__ out, const int32_t *__restrict__ slot_atom,
                             int n_seg) {
  __shared__ double tile[12][65];
  const int g = blockIdx.x, n0 = blockIdx.y * 64;
  for (int idx = threadIdx.x; idx < 64 * 12; idx += blockDim.x) {
    const int k = idx / 12, d = idx - k * 12;
    if (n0 + k < n_seg) tile[d][k] = in[((long long)g * n_seg + n0 + k) * 12 + d];
  }
  __syncthreads();
  for (int idx = threadIdx.x; idx < 64 * 12; idx += blockDim.x) {
    const int d = idx / 64, k = idx - d * 64;
    const int at = slot_atom[4 * g + d / 3];
    if (at >= 0 && n0 + k < n_seg) out[(3LL * at + d % 3) * n_seg + n0 + k] = tile[d][k];
  }
}

int qhp_qtb_export_segment(qhp_system *s, const double *in, double *out) {
  const dim3 grid((unsigned)(s->n_slots / 4), (unsigned)((s->n_seg + 63) / 64));
  k_seg_export<<<grid, 256, 0, s->stream>>>(in, out, s->slot_atom, s->n_seg);
  QHP_LAUNCH_OK(s);
  return QHP_OK;
}

__global__ void k_fill(double *p, long long n, double v) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = v;
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
int qhp_qtb_init(qhp_system *s) {
  const int ns = s->n_seg, nf = ns + 1, nt = s->nt, N = s->N;
  QHP_CUDA_OK(s, cudaMalloc(&s->gamma, sizeof(double) * nt * nf));
  QHP_CUDA_OK(s, cudaMalloc(&s->Hf, sizeof(double) * nt * nf));
  QHP_CUDA_OK(s, cudaMalloc(&s->hk, sizeof(double) * nt * 2 * ns));
  QHP_CUDA_OK(s, cudaMalloc(&s->H4, sizeof(double) * 2 * nt * 4 * ns));
  QHP_CUDA_OK(s, cudaMalloc(&s->Cvv, sizeof(double) * nt * nf));
  QHP_CUDA_OK(s, cudaMalloc(&s->CvF, sizeof(double) * nt * nf));
  QHP_CUDA_OK(s, cudaMalloc(&s->tw, sizeof(double) * 2 * 4 * ns));
  // segment slots: atoms sorted by type, every type padded to whole groups of 4 slots
  std::vector<int32_t> type_host(N), seg_slot(N), slot_atom;
  QHP_CUDA_OK(s, cudaMemcpy(type_host.data(), s->dt_.type, sizeof(int32_t) * N, cudaMemcpyDeviceToHost));
  s->type_start.assign(nt + 1, 0);
  std::vector<double> ndof(nt);
  for (int z = 0; z < nt; ++z) {
    s->type_start[z] = (int)slot_atom.size();
    int cnt = 0;
    for (int a = 0; a < N; ++a)
      if (type_host[a] == z) { seg_slot[a] = (int32_t)slot_atom.size(); slot_atom.push_back(a); ++cnt; }
    while (slot_atom.size() % 4) slot_atom.push_back(-1);
    ndof[z] = 3.0 * cnt;
  }
  s->type_start[nt] = (int)slot_atom.size();
  s->n_slots = (int)slot_atom.size();
  QHP_CUDA_OK(s, cudaMalloc(&s->seg_slot, sizeof(int32_t) * N));
  QHP_CUDA_OK(s, cudaMemcpy(s->seg_slot, seg_slot.data(), sizeof(int32_t) * N, cudaMemcpyHostToDevice));
  QHP_CUDA_OK(s, cudaMalloc(&s->slot_atom, sizeof(int32_t) * slot_atom.size()));
  QHP_CUDA_OK(s, cudaMemcpy(s->slot_atom, slot_atom.data(), sizeof(int32_t) * slot_atom.size(), cudaMemcpyHostToDevice));
  const size_t seg_bytes = sizeof(double) * 3 * (size_t)s->n_slots * ns;
  if (cudaMalloc(&s->Fc, seg_bytes) != cudaSuccess || cudaMalloc(&s->vseg, seg_bytes) != cudaSuccess) {
    s->err = "adQTB segment buffers: out of device memory";
    return QHP_ENOMEM;
  }
  QHP_CUDA_OK(s, cudaMemsetAsync(s->Fc, 0, seg_bytes, s->stream));
  QHP_CUDA_OK(s, cudaMemsetAsync(s->vseg, 0, seg_bytes, s->stream));
  k_twiddle<<<(4 * ns + 255) / 256, 256, 0, s->stream>>>((double2 *)s->tw, 4 * ns);
  QHP_LAUNCH_OK(s);
  k_fill<<<(nt * nf + 255) / 256, 256, 0, s->stream>>>(s->gamma, (long long)nt * nf, s->th.gamma0);
  QHP_LAUNCH_OK(s);
  // spectra CTAs walk runs of <= chunk slot groups of one type: about two CTAs per SM in all
  int sms = 148;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, s->device);
  const int n_groups = s->n_slots / 4;
  int chunk = (n_groups + 2 * sms - 1) / (2 * sms);
  if (chunk < 1) chunk = 1;
  std::vector<int32_t> tab;
  for (int z = 0; z < nt; ++z)
    for (int b = s->type_start[z] / 4; b < s->type_start[z + 1] / 4; b += chunk) {
      tab.push_back(z); tab.push_back(b); tab.push_back(std::min(b + chunk, s->type_start[z + 1] / 4));
    }
  s->n_spec_cta = (int)tab.size() / 3;
  QHP_CUDA_OK(s, cudaMalloc(&s->spec_cta, sizeof(int32_t) * std::max<size_t>(tab.size(), 1)));
  QHP_CUDA_OK(s, cudaMemcpy(s->spec_cta, tab.data(), sizeof(int32_t) * tab.size(), cudaMemcpyHostToDevice));
  QHP_CUDA_OK(s, cudaMalloc(&s->spec_part, sizeof(double) * (size_t)s->n_spec_cta * 2 * nf + sizeof(double) * nt));
  // per-type DOF counts live behind the partials
  QHP_CUDA_OK(s, cudaMemcpy(s->spec_part + (size_t)s->n_spec_cta * 2 * nf, ndof.data(), sizeof(double) * nt, cudaMemcpyHostToDevice));
  return QHP_OK;
}

// Q3 + Q2 + Q4 for segment `seg` with the current gamma_z
int qhp_qtb_generate(qhp_system *s, int64_t seg) {
  const int ns = s->n_seg, nf = ns + 1, nt = s->nt;
  k_qtb_filter<<<(nt * nf + 127) / 128, 128, 0, s->stream>>>(nt, ns, s->dt, QHP_KB * s->T, s->th.classical, s->dt_.mass, s->gamma, s->kappa, s->Hf);
  QHP_LAUNCH_OK(s);
  k_qtb_kernel<<<(nt * 2 * ns + 127) / 128, 128, 0, s->stream>>>(nt, ns, s->Hf, s->hk);
  QHP_LAUNCH_OK(s);
  k_qtb_spectrum4<<<(nt * 4 * ns + 127) / 128, 128, 0, s->stream>>>(nt, ns, s->hk, (double2 *)s->H4);
  QHP_LAUNCH_OK(s);
  const int n4 = 4 * ns;
  const size_t smem = sizeof(double2) * FPAD_LEN(n4) + sizeof(double) * 2 * 3 * ns;
  QHP_CUDA_OK(s, cudaFuncSetAttribute(k_qtb_noise, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_qtb_noise<<<s->n_slots / 2, fft_threads(n4), smem, s->stream>>>(ns, s->th.seed, seg, s->slot_atom, s->dt_.type, (const double2 *)s->H4,
                                                                   (const double2 *)s->tw, s->Fc);
  QHP_LAUNCH_OK(s);
  s->fc_segment = seg;
  return QHP_OK;
}

// Q5-Q7 at the end of a segment
int qhp_qtb_adapt(qhp_system *s) {
  const int ns = s->n_seg, nf = ns + 1, nt = s->nt, nk = 2 * ns;
  // DOFs transformed side by side: 3 (n_seg <= 1024: 384 threads), else 1 (256 threads); every kernel that calls
  // the shared-memory FFT keeps <= 512 threads per CTA so that the radix-16 butterflies stay in registers
  const int dpr = ns <= 1024 ? 3 : 1;
  const size_t smem = sizeof(double2) * 2 * dpr * (nk + 1) + sizeof(double) * 2 * nf;      // two buffers
  if (dpr == 3) {
    QHP_CUDA_OK(s, cudaFuncSetAttribute(k_qtb_spectra<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_qtb_spectra<3><<<s->n_spec_cta, 3 * (nk / 8 < 32 ? 32 : nk / 8), smem, s->stream>>>(ns, s->spec_cta, s->vseg, s->Fc, (const double2 *)s->tw, 4 * ns, s->spec_part);
  } else {
    QHP_CUDA_OK(s, cudaFuncSetAttribute(k_qtb_spectra<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_qtb_spectra<1><<<s->n_spec_cta, (nk / 8 < 32 ? 32 : nk / 8), smem, s->stream>>>(ns, s->spec_cta, s->vseg, s->Fc, (const double2 *)s->tw, 4 * ns, s->spec_part);
  }
  QHP_LAUNCH_OK(s);
  k_qtb_reduce<<<(nt * nf + 127) / 128, 128, 0, s->stream>>>(nt, ns, s->n_spec_cta, s->spec_cta, s->spec_part,
                                                           s->spec_part + (size_t)s->n_spec_cta * 2 * nf, s->dt, s->Cvv, s->CvF);
  QHP_LAUNCH_OK(s);
  if (s->th.a_gamma != 0.0) {
    k_qtb_adapt<<<nt, 256, 0, s->stream>>>(ns, s->dt_.mass, s->th.gamma0, s->th.a_gamma, s->th.gamma_min_frac, s->Cvv, s->CvF, s->gamma,
                                           s->ratio_tau);
    QHP_LAUNCH_OK(s);
  }
  if (s->ratio_tau) {
    k_qtb_adapt_ratio<<<(nt * nf + 127) / 128, 128, 0, s->stream>>>(nt, ns, s->dt_.mass, s->th.gamma0, s->th.gamma_min_frac, s->dt,
                                                                    s->ratio_tau, s->ratio_started ? 0 : 1, s->Cvv, s->CvF,
                                                                    s->ratio_avv, s->ratio_avf, s->gamma);
    QHP_LAUNCH_OK(s);
    s->ratio_started = true;
  }
  return QHP_OK;
}
