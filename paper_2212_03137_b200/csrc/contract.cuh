// contract.cuh -- contraction (Eq. 20) of the current normal modes for one DOF; shared by k_contract
// (nm_kernels.cu) and the fused rebuild kernel (cells.cu).
#pragma once
#include "qhp_internal.cuh"

struct BoxArg { double box[3], inv_box[3]; };

// mode 0: write pos4 in slot order (after a list rebuild also cent4 = sorted centroids + molecule id, the fp32
// copy, cref = centroids in atom order, pos4.w = type); mode 1: write xc_out [Pc][N][3] in atom order (parity hook).
__device__ __forceinline__ void qhp_contract_dof(const BoxArg &bx, const double *__restrict__ Q, int N, int Pc,
                                                 const double *__restrict__ Tc, const int32_t *__restrict__ rank,
                                                 const int32_t *__restrict__ type, const int32_t *__restrict__ molid,
                                                 double *pos4, double *cent4, double *cref, double *xc_out, int mode,
                                                 double thresh2, long long *counters, long long d) {
  const long long ND = 3LL * N;
  const int atom = (int)(d / 3), c = (int)(d % 3);
  const double spc = sqrt((double)Pc);
  const long long slot = rank ? rank[atom] : atom;
  for (int j = 0; j < Pc; ++j) {
    double s = 0.0;
    for (int n = 0; n < Pc; ++n) s += Tc[j * Pc + n] * Q[n * ND + d];
    const double xc = spc * s;
    if (mode == 0) {
      // a list built on the centroids can only cover beads closer than skin/2 to their centroid: the
      // thread of component 0 tests the NORM of the bead's offset (all three components)
      if (cent4 && c == 0) {
        double n2 = (xc - Q[d]) * (xc - Q[d]);
        for (int cc = 1; cc < 3; ++cc) {
          double sc = 0.0;
          for (int n = 0; n < Pc; ++n) sc += Tc[j * Pc + n] * Q[n * ND + d + cc];
          n2 += (spc * sc - Q[d + cc]) * (spc * sc - Q[d + cc]);
        }
        if (n2 > thresh2) counters[6] = 1;
      }
      pos4[((long long)j * N + slot) * 4 + c] = xc;
      if (c == 0) reinterpret_cast<long long *>(pos4)[((long long)j * N + slot) * 4 + 3] = type[atom];
    } else {
      xc_out[(long long)j * ND + d] = xc;
    }
  }
  if (mode == 0 && cent4) {
    const double q0 = Q[d];
    cent4[slot * 4 + c] = q0;
    if (c == 0) reinterpret_cast<long long *>(cent4)[slot * 4 + 3] = molid[atom];
    // single-precision copy, wrapped into [0, L), for the pre-test of the list build (cells.cu);
    // w = molecule id | atom type << 28 (the list entries of the staged pair kernel carry the type)
    float *centf = reinterpret_cast<float *>(cent4 + 4LL * N);
    centf[slot * 4 + c] = (float)(q0 - bx.box[c] * floor(q0 * bx.inv_box[c]));
    if (c == 0) reinterpret_cast<int *>(centf)[slot * 4 + 3] = molid[atom] | (type[atom] << 28);
    cref[d] = q0;
  }
}
