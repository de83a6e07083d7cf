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
__device__ __forceinline__ void fft_pass(double2 *buf, int n, int Ns, const double2 *__restrict__ tw, int tw_n, int t) {
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
        for (int u = 0; u < R; ++u) v[q * R + u] = buf[j + u * nb];
        if (k) {
          const double2 w1 = twiddle(tw, tw_n, k, Ns * R, SG);
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
          for (int d = 0; d < 4; ++d) buf[j0[0] + (c + 4 * d) * Ns] = v[4 * c + d];
      }
    } else {
#pragma unroll
      for (int q = 0; q < G; ++q)
        if (j0[q] >= 0) {
          if (R == 4) {
            dft4<SG>(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
#pragma unroll
            for (int u = 0; u < 4; ++u) buf[j0[q] + u * Ns] = v[4 * q + u];
          } else {
            const double2 x0 = v[2 * q], x1 = v[2 * q + 1];
            buf[j0[q]] = make_double2(x0.x + x1.x, x0.y + x1.y);
            buf[j0[q] + Ns] = make_double2(x0.x - x1.x, x0.y - x1.y);
          }
        }
    }
  }
  __syncthreads();
}

// In-place Stockham FFT of buf[0..n) by blockDim.x >= max(n/16, 1) threads (all threads of the CTA
// must call).  sign = -1 forward, +1 inverse (unnormalised).  Result in natural order.
template <int SG>
__device__ __forceinline__ void fft_smem_sg(double2 *buf, int n, const double2 *__restrict__ tw, int tw_n, int t) {
  int Ns = 1;
  while (n / Ns >= 16 && ((n / Ns) & 15) == 0) { fft_pass<16, SG>(buf, n, Ns, tw, tw_n, t); Ns <<= 4; }
  while (((n / Ns) & 3) == 0 && Ns < n) { fft_pass<4, SG>(buf, n, Ns, tw, tw_n, t); Ns <<= 2; }
  while (Ns < n) { fft_pass<2, SG>(buf, n, Ns, tw, tw_n, t); Ns <<= 1; }
}
// t: index of the calling thread inside its FFT (threads t >= max(n/16, 1) only take part in the barriers);
// several FFTs of the same length can run side by side in one CTA on different buffers.
__device__ __noinline__ void fft_smem(double2 *buf, int n, int sign, const double2 *__restrict__ tw, int tw_n, int t) {
  if (sign < 0) fft_smem_sg<-1>(buf, n, tw, tw_n, t);
  else fft_smem_sg<1>(buf, n, tw, tw_n, t);
}

__global__ void k_twiddle(double2 *tw, int n) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n) return;
  double s, c;
  sincospi(-2.0 * (double)m / (double)n, &s, &c);
  tw[m] = make_double2(c, s);
}

__global__ void __launch_bounds__(512) k_fft_batch(double2 *data, int n, int sign, const double2 *__restrict__ tw, int tw_n) {
  extern __shared__ double2 fbuf[];
  double2 *d = data + (long long)blockIdx.x * n;
  for (int k = threadIdx.x; k < n; k += blockDim.x) fbuf[k] = d[k];
  __syncthreads();
  fft_smem(fbuf, n, sign, tw, tw_n, threadIdx.x);
  for (int k = threadIdx.x; k < n; k += blockDim.x) d[k] = fbuf[k];
}

static int fft_threads(int n) { return n / 16 < 32 ? 32 : n / 16; }

int qhp_fft_launch(double *data, int n, int64_t batch, int sign, const double *tw, int tw_n, cudaStream_t st) {
  const size_t smem = sizeof(double2) * (size_t)n;
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

// ---------------------------------------------------------------------------------------------
// Q2 + Q4: one CTA per atom.  (x, y) white noise of the atom go through one complex FFT (the
// kernel h is real, so real and imaginary parts are filtered independently), z through a second.
//   F_c[dof][n] = sum_k h_z[k] r(dof, seg*n_seg + n - k + n_seg),  n = 0..n_seg-1
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256, 2) k_qtb_noise(int n_seg, long long ND, unsigned long long seed, long long seg, const int32_t *__restrict__ type,
                            const double2 *__restrict__ H4, const double2 *__restrict__ tw, double *Fc) {
  extern __shared__ double2 nbuf[];
  const int nf = 4 * n_seg, nw = 3 * n_seg;
  double *zb = reinterpret_cast<double *>(nbuf + nf);
  const int atom = blockIdx.x, t = threadIdx.x;
  const double2 *Hz = H4 + (long long)type[atom] * nf;
  for (int m = t; m < nf; m += blockDim.x) {
    if (m < nw) {
      double z[3];
      qhp_normals3(seed, (uint32_t)atom, 0u, QHP_TAG_QTB, (uint64_t)(seg * n_seg + m), z);
      nbuf[m] = make_double2(z[0], z[1]);
      zb[m] = z[2];
    } else {
      nbuf[m] = make_double2(0.0, 0.0);
    }
  }
  const double inv = 1.0 / (double)nf;
  double fx[4] = {0.0, 0.0, 0.0, 0.0}, fy[4] = {0.0, 0.0, 0.0, 0.0};   // 4 blockDim.x >= n_seg: samples n = t + u blockDim.x
  for (int pass = 0; pass < 2; ++pass) {
    __syncthreads();
    fft_smem(nbuf, nf, -1, tw, nf, t);
    for (int q = t; q < nf; q += blockDim.x) nbuf[q] = cmul(nbuf[q], Hz[q]);
    __syncthreads();
    fft_smem(nbuf, nf, +1, tw, nf, t);
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int n = t + u * blockDim.x;
      if (n < n_seg) {
        const double2 y = nbuf[n + 2 * n_seg];
        if (pass == 0) { fx[u] = y.x * inv; fy[u] = y.y * inv; }
        else {
          // Fc[n][dof] (step-contiguous for the integrator): the three components of one sample together
          double *out = Fc + (long long)n * ND + 3LL * atom;
          out[0] = fx[u]; out[1] = fy[u]; out[2] = y.x * inv;
        }
      }
    }
    if (pass == 0) {
      __syncthreads();
      for (int m = t; m < nf; m += blockDim.x) nbuf[m] = make_double2(m < nw ? zb[m] : 0.0, 0.0);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Q5 + Q6: spectra.  One CTA walks a run of atoms of one type; v and F_c of a DOF are the real and
// imaginary part of one zero-padded N_k-point transform.  Per-CTA sums -> fixed-order reduction.
// ---------------------------------------------------------------------------------------------
// One CTA = 3 groups of max(n_k/16, 32) threads; group c transforms DOF c of the current atom (v and
// F_c as real and imaginary part of one zero-padded n_k-point FFT).  Every thread accumulates its own
// frequency bins in registers over all atoms of the CTA's run; the three groups are combined once at
// the end in a fixed order.  SPEC_BINS bounds (n_seg + 1) / group size (n_seg <= 1024: 1025 / 128).
#define SPEC_BINS 9
__global__ void __launch_bounds__(384, 2) k_qtb_spectra(int n_seg, long long ND, const int32_t *__restrict__ cta_tab, const int32_t *__restrict__ atoms,
                              const double *__restrict__ vseg, const double *__restrict__ Fc,
                              const double2 *__restrict__ tw, int tw_n, double *part) {
  extern __shared__ double2 sbuf_all[];
  const int nk = 2 * n_seg, nf = n_seg + 1, gsz = blockDim.x / 3;
  const int c = threadIdx.x / gsz, t = threadIdx.x - c * gsz;
  double2 *sbuf = sbuf_all + (size_t)c * nk;
  double avv[SPEC_BINS], avf[SPEC_BINS];
#pragma unroll
  for (int m = 0; m < SPEC_BINS; ++m) { avv[m] = 0.0; avf[m] = 0.0; }
  const int b = cta_tab[3 * blockIdx.x + 1], e = cta_tab[3 * blockIdx.x + 2];
  for (int ia = b; ia < e; ++ia) {
    const long long d = 3LL * atoms[ia] + c;
    for (int n = t; n < nk; n += gsz)
      sbuf[n] = (n < n_seg) ? make_double2(vseg[(long long)n * ND + d], Fc[(long long)n * ND + d]) : make_double2(0.0, 0.0);
    __syncthreads();
    fft_smem(sbuf, nk, -1, tw, tw_n, t);
#pragma unroll
    for (int m = 0; m < SPEC_BINS; ++m) {
      const int j = t + m * gsz;
      if (j < nf) {
        const double2 A = sbuf[j], Zm = sbuf[(nk - j) & (nk - 1)];
        const double vx = 0.5 * (A.x + Zm.x), vy = 0.5 * (A.y - Zm.y);     // V_j
        const double px = 0.5 * (A.y + Zm.y), py = -0.5 * (A.x - Zm.x);    // Phi_j
        avv[m] += vx * vx + vy * vy;
        avf[m] += vx * px + vy * py;
      }
    }
    __syncthreads();
  }
  // combine the three groups: (x + y) + z per bin
  double *red = reinterpret_cast<double *>(sbuf_all);          // [3][2][nf]
#pragma unroll
  for (int m = 0; m < SPEC_BINS; ++m) {
    const int j = t + m * gsz;
    if (j < nf) { red[(c * 2) * nf + j] = avv[m]; red[(c * 2 + 1) * nf + j] = avf[m]; }
  }
  __syncthreads();
  double *o = part + (long long)blockIdx.x * 2 * nf;
  for (int j = threadIdx.x; j < nf; j += blockDim.x) {
    o[j] = (red[j] + red[2 * nf + j]) + red[4 * nf + j];
    o[nf + j] = (red[nf + j] + red[3 * nf + j]) + red[5 * nf + j];
  }
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

// parity hook: internal [n_seg][3N] -> documented [3N][n_seg]
__global__ void k_seg_transpose(const double *__restrict__ in, double *__restrict__ out, long long ND, int n_seg) {
  __shared__ double tile[32][33];
  const long long d0 = (long long)blockIdx.x * 32;
  const int n0 = blockIdx.y * 32;
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    const long long d = d0 + threadIdx.x;
    const int n = n0 + r;
    tile[r][threadIdx.x] = (d < ND && n < n_seg) ? in[n * ND + d] : 0.0;
  }
  __syncthreads();
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    const long long d = d0 + r;
    const int n = n0 + threadIdx.x;
    if (d < ND && n < n_seg) out[d * n_seg + n] = tile[threadIdx.x][r];
  }
}

int qhp_qtb_export_segment(qhp_system *s, const double *in, double *out) {
  const long long ND = 3LL * s->N;
  const dim3 grid((unsigned)((ND + 31) / 32), (unsigned)((s->n_seg + 31) / 32)), block(32, 8);
  k_seg_transpose<<<grid, block, 0, s->stream>>>(in, out, ND, s->n_seg);
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
  const size_t seg_bytes = sizeof(double) * 3 * (size_t)N * ns;
  QHP_CUDA_OK(s, cudaMalloc(&s->gamma, sizeof(double) * nt * nf));
  QHP_CUDA_OK(s, cudaMalloc(&s->Hf, sizeof(double) * nt * nf));
  QHP_CUDA_OK(s, cudaMalloc(&s->hk, sizeof(double) * nt * 2 * ns));
  QHP_CUDA_OK(s, cudaMalloc(&s->H4, sizeof(double) * 2 * nt * 4 * ns));
  QHP_CUDA_OK(s, cudaMalloc(&s->Cvv, sizeof(double) * nt * nf));
  QHP_CUDA_OK(s, cudaMalloc(&s->CvF, sizeof(double) * nt * nf));
  QHP_CUDA_OK(s, cudaMalloc(&s->tw, sizeof(double) * 2 * 4 * ns));
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
  // atoms grouped by type; spectra CTAs walk runs of <= chunk atoms of one type
  std::vector<int32_t> by_type, type_host(N);
  QHP_CUDA_OK(s, cudaMemcpy(type_host.data(), s->dt_.type, sizeof(int32_t) * N, cudaMemcpyDeviceToHost));
  s->type_start.assign(nt + 1, 0);
  for (int z = 0; z < nt; ++z) {
    s->type_start[z] = (int)by_type.size();
    for (int a = 0; a < N; ++a) if (type_host[a] == z) by_type.push_back(a);
  }
  s->type_start[nt] = (int)by_type.size();
  int chunk = (N + 148 * 4 - 1) / (148 * 4);
  if (chunk < 1) chunk = 1;
  std::vector<int32_t> tab;
  std::vector<double> ndof(nt);
  for (int z = 0; z < nt; ++z) {
    ndof[z] = 3.0 * (s->type_start[z + 1] - s->type_start[z]);
    for (int b = s->type_start[z]; b < s->type_start[z + 1]; b += chunk) {
      tab.push_back(z); tab.push_back(b); tab.push_back(std::min(b + chunk, s->type_start[z + 1]));
    }
  }
  s->n_spec_cta = (int)tab.size() / 3;
  QHP_CUDA_OK(s, cudaMalloc(&s->atoms_by_type, sizeof(int32_t) * N));
  QHP_CUDA_OK(s, cudaMemcpy(s->atoms_by_type, by_type.data(), sizeof(int32_t) * N, cudaMemcpyHostToDevice));
  QHP_CUDA_OK(s, cudaMalloc(&s->spec_cta, sizeof(int32_t) * tab.size()));
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
  const size_t smem = sizeof(double2) * n4 + sizeof(double) * 3 * ns;
  QHP_CUDA_OK(s, cudaFuncSetAttribute(k_qtb_noise, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_qtb_noise<<<s->N, fft_threads(n4), smem, s->stream>>>(ns, 3LL * s->N, s->th.seed, seg, s->dt_.type, (const double2 *)s->H4,
                                                         (const double2 *)s->tw, s->Fc);
  QHP_LAUNCH_OK(s);
  s->fc_segment = seg;
  return QHP_OK;
}

// Q5-Q7 at the end of a segment
int qhp_qtb_adapt(qhp_system *s) {
  const int ns = s->n_seg, nf = ns + 1, nt = s->nt, nk = 2 * ns;
  const size_t smem = sizeof(double2) * 3 * nk;
  QHP_CUDA_OK(s, cudaFuncSetAttribute(k_qtb_spectra, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_qtb_spectra<<<s->n_spec_cta, 3 * fft_threads(nk), smem, s->stream>>>(ns, 3LL * s->N, s->spec_cta, s->atoms_by_type, s->vseg, s->Fc,
                                                                        (const double2 *)s->tw, 4 * ns, s->spec_part);
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
