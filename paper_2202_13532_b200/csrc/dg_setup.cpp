// Host-side setup of the LGL basis, the 1-D DG operators and the DG->Fourier tensor.
// Written from PAPER.md (arXiv 2202.13532) Section 5; long double throughout, rounded once.
// Deliberately uses Eq. 53 (Lagrange-derivative form) for Upsilon where the test oracle uses
// Eq. 57 (Legendre-sum form), and its own spherical Bessel routine, so the two sides share
// neither code nor formula.
#include "dg_setup.hpp"

#include <algorithm>
#include <cmath>
#include <complex>
#include <stdexcept>

namespace dgsetup {

typedef long double ld;
static const ld PI_L = 3.141592653589793238462643383279502884L;

// P_N(x), P_N'(x), P_{N-1}(x) by the Bonnet recurrence.
static void legendre(int N, ld x, ld& P, ld& dP) {
  ld p0 = 1.0L, p1 = x, d0 = 0.0L, d1 = 1.0L;
  if (N == 0) { P = p0; dP = d0; return; }
  for (int s = 1; s < N; ++s) {
    ld p2 = ((2 * s + 1) * x * p1 - s * p0) / (s + 1);
    ld d2 = d0 + (2 * s + 1) * p1;
    p0 = p1; p1 = p2; d0 = d1; d1 = d2;
  }
  P = p1; dP = d1;
}

Basis1D make_basis(int n, int mass_mode) {
  if (n < 2 || n > 10) throw std::invalid_argument("order must be 2..10");
  Basis1D b;
  b.n = n;
  const int N = n - 1;
  std::vector<ld> xi(n), w(n), PN(n);
  // Eq. 45: interior nodes are the roots of P_N'; Newton with P_N'' from the
  // Legendre ODE, started at the Chebyshev-Lobatto points.
  xi[0] = -1.0L; xi[N] = 1.0L;
  for (int j = 1; j < N; ++j) {
    ld x = -std::cos(PI_L * j / N);
    for (int it = 0; it < 100; ++it) {
      ld P, dP; legendre(N, x, P, dP);
      ld ddP = (2 * x * dP - (ld)N * (N + 1) * P) / (1 - x * x);
      ld dx = dP / ddP;
      x -= dx;
      if (fabsl(dx) < 1e-19L) break;
    }
    xi[j] = x;
  }
  for (int j = 0; j < n / 2; ++j) {            // exact antisymmetry
    ld a = 0.5L * (xi[n - 1 - j] - xi[j]);
    xi[j] = -a; xi[n - 1 - j] = a;
  }
  if (n % 2) xi[n / 2] = 0.0L;
  for (int j = 0; j < n; ++j) {
    ld P, dP; legendre(N, xi[j], P, dP);
    PN[j] = P;
    w[j] = 2.0L / ((ld)n * (n - 1) * P * P);
  }
  // l_j'(xi_k) by the barycentric formula (Eq. 4 differentiated; Eq. 55 is D[k][j] = l_j'(xi_k)).
  std::vector<ld> lam(n, 1.0L);
  for (int j = 0; j < n; ++j)
    for (int k = 0; k < n; ++k) if (k != j) lam[j] /= (xi[j] - xi[k]);
  std::vector<ld> dl(n * n, 0.0L);             // dl[k*n + j] = l_j'(xi_k)
  for (int k = 0; k < n; ++k) {
    ld diag = 0.0L;
    for (int j = 0; j < n; ++j) if (j != k) {
      dl[k * n + j] = (lam[j] / lam[k]) / (xi[k] - xi[j]);
      diag -= dl[k * n + j];
    }
    dl[k * n + k] = diag;
  }
  // P_N'(xi_k): zero at interior LGL nodes, (+-1)^{N+1} N(N+1)/2 at the ends.
  std::vector<ld> dPN(n, 0.0L);
  dPN[N] = 0.5L * N * (N + 1);
  dPN[0] = ((N + 1) % 2 == 0 ? 1.0L : -1.0L) * 0.5L * N * (N + 1);
  b.xi.resize(n); b.w.resize(n); b.ups.assign(n * n, 0.0); b.lift.assign(n * 2, 0.0);
  b.xi_ld = xi; b.w_ld = w;
  b.dmat.resize(n * n);
  for (int i = 0; i < n * n; ++i) b.dmat[i] = (double)dl[i];      // (D f)_j = sum_k l_k'(xi_j) f_k
  for (int j = 0; j < n; ++j) { b.xi[j] = (double)xi[j]; b.w[j] = (double)w[j]; }
  for (int j = 0; j < n; ++j) {
    for (int k = 0; k < n; ++k) {
      // Eq. 53: Ups[j][k] = (w_k/w_j) l_j'(xi_k) + (n/2) w_k P_N(xi_j) P_N'(xi_k)
      ld v = (w[k] / w[j]) * dl[k * n + j];
      if (mass_mode == 0) v += 0.5L * n * w[k] * PN[j] * dPN[k];
      b.ups[j * n + k] = (double)v;
    }
    // Eq. 54: Xi[j][face] = delta_{j,face}/w_j + (n/2) P_N(xi_j) P_N(xi_face)
    ld vL = (j == 0 ? 1.0L / w[0] : 0.0L), vR = (j == N ? 1.0L / w[N] : 0.0L);
    if (mass_mode == 0) { vL += 0.5L * n * PN[j] * PN[0]; vR += 0.5L * n * PN[j] * PN[N]; }
    b.lift[j * 2 + 0] = (double)vL;
    b.lift[j * 2 + 1] = (double)vR;
  }
  return b;
}

// Spherical Bessel j_0..j_{smax}(z) by Miller's downward recurrence, normalised with the larger of
// the closed forms j_0 = sin z / z, j_1 = sin z / z^2 - cos z / z (stable for every z > 0, unlike
// the upward recurrence for z < s).
static void spherical_bessel(int smax, ld z, ld* out) {
  if (z == 0.0L) { out[0] = 1.0L; for (int s = 1; s <= smax; ++s) out[s] = 0.0L; return; }
  if (fabsl(z) < 1e-3L) {                       // leading series terms; error O(z^4) relative
    ld term = 1.0L;
    for (int s = 0; s <= smax; ++s) {
      if (s > 0) term *= z / (2 * s + 1);
      ld a = z * z / 2;
      out[s] = term * (1.0L - a / (2 * s + 3) + a * a / (2.0L * (2 * s + 3) * (2 * s + 5))
                       - a * a * a / (6.0L * (2 * s + 3) * (2 * s + 5) * (2 * s + 7)));
    }
    return;
  }
  int start = smax + 30 + (int)(1.5L * fabsl(z));
  std::vector<ld> t(start + 2, 0.0L);
  t[start + 1] = 0.0L; t[start] = 1e-280L;
  for (int s = start; s >= 1; --s) {
    t[s - 1] = (2 * s + 1) / z * t[s] - t[s + 1];
    if (fabsl(t[s - 1]) > 1e250L) for (int q = s - 1; q <= start; ++q) t[q] *= 1e-250L;
  }
  ld j0 = sinl(z) / z, j1 = sinl(z) / (z * z) - cosl(z) / z;
  ld scale = (fabsl(j0) >= fabsl(j1)) ? j0 / t[0] : j1 / t[1];
  for (int s = 0; s <= smax; ++s) out[s] = t[s] * scale;
}

void make_fourier(const Basis1D& b, int nelem, double lo, double hi, int pmax,
                  std::vector<double>& T, std::vector<double>& S, std::vector<double>& x,
                  std::vector<double>* AD, std::vector<double>* W, bool dense) {
  const int n = b.n, G = nelem * n, P1 = pmax + 1;
  const ld L = (ld)hi - (ld)lo, dx = L / nelem;
  T.clear(); S.clear();
  if (dense) {
    T.assign((size_t)2 * P1 * G, 0.0);
    S.assign((size_t)G * 2 * P1, 0.0);
  }
  x.resize(G);
  std::vector<ld> xi(n), w(n), Ps(n * n);      // Ps[s*n + j] = P_s(xi_j)
  for (int j = 0; j < n; ++j) { xi[j] = b.xi_ld[j]; w[j] = b.w_ld[j]; }
  for (int j = 0; j < n; ++j) {
    ld p0 = 1.0L, p1 = xi[j];
    Ps[0 * n + j] = p0; if (n > 1) Ps[1 * n + j] = p1;
    for (int s = 1; s < n - 1; ++s) {
      ld p2 = ((2 * s + 1) * xi[j] * p1 - s * p0) / (s + 1);
      Ps[(s + 1) * n + j] = p2; p0 = p1; p1 = p2;
    }
  }
  for (int m = 0; m < nelem; ++m)
    for (int j = 0; j < n; ++j)
      x[m * n + j] = (double)((ld)lo + (m + 0.5L) * dx + 0.5L * dx * xi[j]);

  // Per mode p: node factor of Eq. 63, w_j sum_s gamma_s^{-1} (-i)^s P_s(xi_j) j_s(k_p dx/2); the phase
  // e^{i k_p lo}; and the in-element phases e^{i k_p (dx/2) xi_j}.
  std::vector<ld> nre((size_t)P1 * n), nim((size_t)P1 * n), pjc((size_t)P1 * n), pjs((size_t)P1 * n), plc(P1), pls(P1);
#pragma omp parallel for schedule(static)
  for (int p = 0; p <= pmax; ++p) {
    const ld kp = 2 * PI_L * p / L;
    std::vector<ld> js(n);
    spherical_bessel(n - 1, kp * dx / 2, js.data());
    for (int j = 0; j < n; ++j) {
      ld re = 0.0L, im = 0.0L;
      for (int s = 0; s < n; ++s) {
        ld ginv = (s < n - 1) ? (2 * s + 1) / 2.0L : (n - 1) / 2.0L;      // 1/gamma_s, Eq. 46
        ld v = ginv * Ps[s * n + j] * js[s];
        switch (s & 3) {                        // (-i)^s = 1, -i, -1, i
          case 0: re += v; break;
          case 1: im -= v; break;
          case 2: re -= v; break;
          default: im += v; break;
        }
      }
      nre[(size_t)p * n + j] = re * w[j]; nim[(size_t)p * n + j] = im * w[j];
      pjc[(size_t)p * n + j] = cosl(kp * 0.5L * dx * xi[j]);
      pjs[(size_t)p * n + j] = sinl(kp * 0.5L * dx * xi[j]);
    }
    plc[p] = cosl(kp * (ld)lo); pls[p] = sinl(kp * (ld)lo);
  }
  // e^{i k_p (xbar_m - lo)} = e^{i 2 pi p (2m+1) / (2 nelem)}: the argument is reduced exactly in integers.
  auto mid_phase = [&](int p, int m, ld& c, ld& s) {
    long long r = ((long long)p * (2LL * m + 1)) % (2LL * nelem);
    ld ang = PI_L * (ld)r / (ld)nelem;
    c = cosl(ang); s = sinl(ang);
  };
#pragma omp parallel for schedule(static)
  for (int p = 0; p <= (dense ? pmax : -1); ++p) {
    for (int m = 0; m < nelem; ++m) {
      ld c0, s0; mid_phase(p, m, c0, s0);
      // e^{-i k xbar} * (dx/L)
      const ld c = (c0 * plc[p] - s0 * pls[p]) * (dx / L), sgn = -(s0 * plc[p] + c0 * pls[p]) * (dx / L);
      for (int j = 0; j < n; ++j) {
        const size_t g = (size_t)m * n + j;
        const ld re = nre[(size_t)p * n + j], im = nim[(size_t)p * n + j];
        T[((size_t)(2 * p) * G) + g] = (double)(c * re - sgn * im);          // Eq. 63, real part
        T[((size_t)(2 * p + 1) * G) + g] = (double)(c * im + sgn * re);      // imaginary part
      }
    }
  }
  // Tables of the FFT-factorised form (dg_kernels_fft.cuh), equal-width elements, p fastest:
  //   rows 0..n/2-1   B_p^j = node factor of Eq. 63 (B_p^{n-1-j} = conj B_p^j: the LGL nodes are symmetric)
  //   rows n/2..n-1   u_p^j / (k_p N),  u_p^j = e^{i k_p xi_j dx/2}   (u_p^{n-1-j} = conj u_p^j; zero at p = 0)
  //   row  n          a_p   = e^{-i phi_p} / N,  phi_p = k_p lo + pi p / N  (the element-centre phase without its
  //                   e^{-2 pi i p m/N} part)
  //   W_k = e^{-2 pi i k/N}.
  if (AD && W) {
    const int NPh = n / 2;
    AD->assign((size_t)P1 * (n + 1) * 2, 0.0);
    W->assign((size_t)(nelem / 2 > 0 ? nelem / 2 : 1) * 2, 0.0);
    for (int k = 0; k < nelem / 2; ++k) {
      (*W)[2 * k] = (double)cosl(2 * PI_L * k / nelem);
      (*W)[2 * k + 1] = (double)(-sinl(2 * PI_L * k / nelem));
    }
#pragma omp parallel for schedule(static)
    for (int p = 0; p <= pmax; ++p) {
      const ld ang = PI_L * (ld)(p % (2 * nelem)) / (ld)nelem;
      const ld cm = cosl(ang), sm = sinl(ang);
      const ld cphi = plc[p] * cm - pls[p] * sm, sphi = pls[p] * cm + plc[p] * sm;
      for (int j = 0; j < NPh; ++j) {
        double* bq = AD->data() + ((size_t)j * P1 + p) * 2;
        bq[0] = (double)nre[(size_t)p * n + j]; bq[1] = (double)nim[(size_t)p * n + j];
        double* uq = AD->data() + ((size_t)(NPh + j) * P1 + p) * 2;
        const ld fk = p ? L / (2 * PI_L * p * nelem) : 0.0L;                 // 1 / (k_p N): Poisson factor of Eq. 71
        uq[0] = (double)(fk * pjc[(size_t)p * n + j]); uq[1] = (double)(fk * pjs[(size_t)p * n + j]);
      }
      double* aq = AD->data() + ((size_t)n * P1 + p) * 2;
      aq[0] = (double)(cphi / nelem); aq[1] = (double)(-sphi / nelem);
    }
  }
  // Synthesis with the Poisson factor folded in (Eq. 71): E = sum_{p>=1} 2 Re( (i c_p / k_p) e^{i k_p x} )
  //   = sum_p (-2/k_p) ( Re c_p sin(k_p x) + Im c_p cos(k_p x) ).
#pragma omp parallel for schedule(static)
  for (int m = 0; m < (dense ? nelem : 0); ++m) {
    for (int p = 1; p <= pmax; ++p) {
      const ld kp = 2 * PI_L * p / L;
      ld c0, s0; mid_phase(p, m, c0, s0);
      const ld c1 = c0 * plc[p] - s0 * pls[p], s1 = s0 * plc[p] + c0 * pls[p];   // e^{i k xbar}
      for (int j = 0; j < n; ++j) {
        const ld cj = pjc[(size_t)p * n + j], sj = pjs[(size_t)p * n + j];
        const ld cth = c1 * cj - s1 * sj, sth = s1 * cj + c1 * sj;
        const size_t g = (size_t)m * n + j;
        S[g * 2 * P1 + 2 * p] = (double)(-2.0L / kp * sth);
        S[g * 2 * P1 + 2 * p + 1] = (double)(-2.0L / kp * cth);
      }
    }
  }
}

// Non-uniform element widths: Eq. 63 with its per-element (Delta x)_m, dense T and S only (the FFT
// factorisation needs equal widths).  edges[0..N] ascending; x periodic with L = edges[N] - edges[0].
void make_fourier_nonuniform(const Basis1D& b, const std::vector<double>& edges, int pmax,
                             std::vector<double>& T, std::vector<double>& S, std::vector<double>& x) {
  const int n = b.n, nelem = (int)edges.size() - 1, G = nelem * n, P1 = pmax + 1;
  const ld lo = edges[0], L = (ld)edges[nelem] - (ld)edges[0];
  T.assign((size_t)2 * P1 * G, 0.0);
  S.assign((size_t)G * 2 * P1, 0.0);
  x.resize(G);
  std::vector<ld> Ps(n * n), xl(G);
  for (int j = 0; j < n; ++j) {
    ld p0 = 1.0L, p1 = b.xi_ld[j];
    Ps[0 * n + j] = p0; if (n > 1) Ps[1 * n + j] = p1;
    for (int s = 1; s < n - 1; ++s) {
      ld p2 = ((2 * s + 1) * b.xi_ld[j] * p1 - s * p0) / (s + 1);
      Ps[(s + 1) * n + j] = p2; p0 = p1; p1 = p2;
    }
  }
  for (int m = 0; m < nelem; ++m)
    for (int j = 0; j < n; ++j) {
      xl[m * n + j] = 0.5L * ((ld)edges[m] + (ld)edges[m + 1]) + 0.5L * ((ld)edges[m + 1] - (ld)edges[m]) * b.xi_ld[j];
      x[m * n + j] = (double)xl[m * n + j];
    }
  // cos, sin of k_p y with the argument reduced in units of the period: p (y - lo)/L mod 1, plus k_p lo
  auto phase = [&](int p, ld y, ld& c, ld& s) {
    ld t = (ld)p * ((y - lo) / L);
    t -= floorl(t);
    const ld ang = 2 * PI_L * t + 2 * PI_L * p * (lo / L);
    c = cosl(ang); s = sinl(ang);
  };
#pragma omp parallel for schedule(dynamic, 4)
  for (int p = 0; p <= pmax; ++p) {
    const ld kp = 2 * PI_L * p / L;
    std::vector<ld> js(n);
    for (int m = 0; m < nelem; ++m) {
      const ld dx = (ld)edges[m + 1] - (ld)edges[m], xbar = 0.5L * ((ld)edges[m] + (ld)edges[m + 1]);
      spherical_bessel(n - 1, kp * dx / 2, js.data());
      ld c0, s0; phase(p, xbar, c0, s0);
      const ld c = c0 * (dx / L), sgn = -s0 * (dx / L);                 // (dx_m / L) e^{-i k xbar_m}
      for (int j = 0; j < n; ++j) {
        ld re = 0.0L, im = 0.0L;
        for (int s = 0; s < n; ++s) {
          const ld ginv = (s < n - 1) ? (2 * s + 1) / 2.0L : (n - 1) / 2.0L;      // 1/gamma_s, Eq. 46
          const ld v = ginv * Ps[s * n + j] * js[s];
          switch (s & 3) { case 0: re += v; break; case 1: im -= v; break; case 2: re -= v; break; default: im += v; break; }
        }
        re *= b.w_ld[j]; im *= b.w_ld[j];
        const size_t g = (size_t)m * n + j;
        T[((size_t)(2 * p) * G) + g] = (double)(c * re - sgn * im);
        T[((size_t)(2 * p + 1) * G) + g] = (double)(c * im + sgn * re);
        if (p > 0) {
          ld cth, sth; phase(p, xl[g], cth, sth);
          S[g * 2 * P1 + 2 * p] = (double)(-2.0L / kp * sth);               // Eq. 71 with -1/(i k_p) folded in
          S[g * 2 * P1 + 2 * p + 1] = (double)(-2.0L / kp * cth);
        }
      }
    }
  }
}

// SSP-RK3 stability limit of the 1-D periodic upwind DG operator (the paper defers its CFL numbers
// to ref. [39]).  For Bloch phase th the element operator (a > 0, unit a, J = 2/dx) is
// A(th) = Ups - Xi_R e_R^T + e^{-i th} Xi_L e_R^T;  the step matrix is R = I + Z + Z^2/2 + Z^3/6 with
// Z = nu * 2 * A.  nu is stable iff rho(R) <= 1 for every th, tested by repeated squaring of R.
typedef std::complex<double> cd;
static void matmul(int n, const std::vector<cd>& A, const std::vector<cd>& B, std::vector<cd>& C) {
  for (int i = 0; i < n; ++i)
    for (int j = 0; j < n; ++j) {
      cd acc = 0;
      for (int k = 0; k < n; ++k) acc += A[i * n + k] * B[k * n + j];
      C[i * n + j] = acc;
    }
}
static bool rk3_stable(const Basis1D& b, double nu, int nphase) {
  const int n = b.n;
  std::vector<cd> Z(n * n), Z2(n * n), Z3(n * n), R(n * n), Tm(n * n);
  for (int q = 0; q <= nphase; ++q) {
    const double th = 3.14159265358979323846 * q / nphase;      // spectrum is symmetric in th
    const cd ph = std::polar(1.0, -th);
    for (int j = 0; j < n; ++j)
      for (int k = 0; k < n; ++k) {
        cd v = b.ups[j * n + k];
        if (k == n - 1) v += -b.lift[j * 2 + 1] + ph * b.lift[j * 2 + 0];
        Z[j * n + k] = 2.0 * nu * v;
      }
    matmul(n, Z, Z, Z2); matmul(n, Z2, Z, Z3);
    for (int i = 0; i < n * n; ++i) R[i] = Z[i] + 0.5 * Z2[i] + Z3[i] / 6.0;
    for (int i = 0; i < n; ++i) R[i * n + i] += 1.0;
    for (int it = 0; it < 24; ++it) {                           // R^(2^24)
      matmul(n, R, R, Tm); R.swap(Tm);
      double mx = 0; for (int i = 0; i < n * n; ++i) mx = std::max(mx, std::abs(R[i]));
      if (mx > 1e6) return false;
      if (mx < 1e-30) break;
    }
  }
  return true;
}
double rk3_cfl_limit(const Basis1D& b) {
  double lo = 0.0, hi = 2.0;
  for (int it = 0; it < 30; ++it) {
    double mid = 0.5 * (lo + hi);
    if (rk3_stable(b, mid, 96)) lo = mid; else hi = mid;
  }
  return lo;
}

}  // namespace dgsetup
