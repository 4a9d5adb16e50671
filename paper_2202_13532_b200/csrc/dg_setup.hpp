// Host-side setup of the LGL basis, DG operators and the DG->Fourier tensor (see dg_setup.cpp).
#pragma once
#include <vector>

namespace dgsetup {

struct Basis1D {
  int n = 0;
  std::vector<double> xi, w;        // LGL nodes / weights on [-1,1]            (Eq. 45)
  std::vector<long double> xi_ld, w_ld;
  std::vector<double> ups;          // Upsilon[j*n + k], reference element      (Eq. 53)
  std::vector<double> lift;         // Xi[j*2 + {0:L,1:R}]                      (Eq. 54)
  std::vector<double> dmat;         // D[j*n + k] = l_k'(xi_j)                  (Eq. 55), strong form Eq. 15
};

Basis1D make_basis(int n, int mass_mode);

// T[(2p+c)*G + g]   : c = 0 real, 1 imaginary part of T_p^{mj} of Eq. 63, g = m*n + j
// S[g*2*(pmax+1) + 2p + c] : synthesis row of Eq. 71 with the Poisson factor -1/(i k_p) folded in,
//                     so that E[g] = sum_{p,c} S[g][2p+c] * c_p[c]; columns of p = 0 are zero.
// x[g]              : node coordinates.
// dense = false     : T and S are left empty (only x and the tables below are built).
// AD, W (optional)  : tables of the FFT-factorised form (even n), AD[(row*P1 + p)*2 + {re,im}]: rows 0..n/2-1 the node
//                     factors B_p^j of Eq. 63, rows n/2..n-1 the in-element phases u_p^j, row n the centre phase a_p;
//                     W[2k + {re,im}] = e^{-2 pi i k / nelem}, k < nelem/2 (see dg_kernels_fft.cuh).
void make_fourier(const Basis1D& b, int nelem, double lo, double hi, int pmax,
                  std::vector<double>& T, std::vector<double>& S, std::vector<double>& x,
                  std::vector<double>* AD = nullptr, std::vector<double>* W = nullptr, bool dense = true);

// The same dense T, S and x for explicitly given element edges (non-uniform widths, Eq. 63 with (Delta x)_m).
void make_fourier_nonuniform(const Basis1D& b, const std::vector<double>& edges, int pmax,
                             std::vector<double>& T, std::vector<double>& S, std::vector<double>& x);

// Largest a*dt/dx for which SSP-RK3 is stable on the 1-D periodic upwind DG operator built from `b`.
double rk3_cfl_limit(const Basis1D& b);

}  // namespace dgsetup
