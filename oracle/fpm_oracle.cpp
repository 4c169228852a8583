// fpm_oracle.cpp -- float64 CPU ORACLE for the FastPM particle-mesh path (TEST INFRASTRUCTURE).
//
// This file is the parity reference for the CUDA library in paper_2010_11847_b200/csrc and the
// timed "cpu_baseline" of bench.py.  It is NOT part of the product path: only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
// It shares no code, header, table or helper with the CUDA path and is written to be checked
// against the paper by eye: plain loops, float64 everywhere, no blocking/fusion/reordering
// beyond what each definition states.  OpenMP only parallelises independent outer loops
// (pencils of the FFT, particles of a gather); paint is serial.
//
// Citations are PAPER.md:LINE (FlowPM, arxiv 2010.11847) and SURVEY.md section 8(c) readings
// R0-R13 (the paper defers most formulas to Feng et al. 2016; every such reading is listed in
// DESIGN.md).  Pins for every function live in tests/test_oracle_*.py ("parity unpinned": none).
//
// Layouts (same as include/fpm.h so inputs can be shared):
//   particles  pos/mom/force : [3][n] planes, float64, mesh-cell units, x in [0, ng)
//   real mesh                : [ng][ng][ng], z fastest
//   k-space                  : [ng][ng][ng/2+1] interleaved (re, im), integer frequency
//                              n_d in (-ng/2, ng/2], omega_d = 2 pi n_d / ng
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

using cd = std::complex<double>;
const double PI = 3.14159265358979323846264338327950288;

inline int64_t wrap_index(int64_t i, int64_t ng) {
  i %= ng;
  return i < 0 ? i + ng : i;
}

// ------------------------------------------------------------------------------------------
// R5  Growth functions (paper silent).  Unknowns y = (D1, G1, D2, G2) with
// G = a^3 E dD/da:   dD/da = G/(a^3 E),  dG1/da = 1.5 Om D1/(a^2 E),
//                    dG2/da = 1.5 Om (D2 - D1^2)/(a^2 E).
// RK4 in ln a from a = 1e-4 with matter-era data D1 = a, D2 = -(3/7) a^2.
// ------------------------------------------------------------------------------------------
inline double E_of_a(double om, double a) { return std::sqrt(om / (a * a * a) + 1.0 - om); }

void growth_rhs(double om, double lna, const double y[4], double dy[4]) {
  const double a = std::exp(lna), E = E_of_a(om, a);
  // d/dlna = a d/da
  dy[0] = a * y[1] / (a * a * a * E);
  dy[1] = a * 1.5 * om * y[0] / (a * a * E);
  dy[2] = a * y[3] / (a * a * a * E);
  dy[3] = a * 1.5 * om * (y[2] - y[0] * y[0]) / (a * a * E);
}

void growth_integrate(double om, double a_end, double y[4]) {
  const double a_ini = 1e-4;
  const int nstep = 20000;
  const double E = E_of_a(om, a_ini);
  y[0] = a_ini;                                   // D1 = a
  y[1] = a_ini * a_ini * a_ini * E * 1.0;         // G1 = a^3 E dD1/da
  y[2] = -3.0 / 7.0 * a_ini * a_ini;              // D2 = -(3/7) a^2
  y[3] = a_ini * a_ini * a_ini * E * (-6.0 / 7.0 * a_ini);
  const double h = (std::log(a_end) - std::log(a_ini)) / nstep;
  double lna = std::log(a_ini);
  for (int s = 0; s < nstep; ++s) {
    double k1[4], k2[4], k3[4], k4[4], t[4];
    growth_rhs(om, lna, y, k1);
    for (int i = 0; i < 4; ++i) t[i] = y[i] + 0.5 * h * k1[i];
    growth_rhs(om, lna + 0.5 * h, t, k2);
    for (int i = 0; i < 4; ++i) t[i] = y[i] + 0.5 * h * k2[i];
    growth_rhs(om, lna + 0.5 * h, t, k3);
    for (int i = 0; i < 4; ++i) t[i] = y[i] + h * k3[i];
    growth_rhs(om, lna + h, t, k4);
    for (int i = 0; i < 4; ++i) y[i] += h / 6.0 * (k1[i] + 2 * k2[i] + 2 * k3[i] + k4[i]);
    lna += h;
  }
}

struct Growth { double D1, f1, D2, f2, E, Gf, gf; };

Growth growth_at(double om, double a) {
  double y[4], y1[4];
  growth_integrate(om, a, y);
  growth_integrate(om, 1.0, y1);
  const double norm = y1[0];                      // D1(1) = 1
  Growth g;
  g.E = E_of_a(om, a);
  g.D1 = y[0] / norm;
  g.D2 = y[2] / (norm * norm);
  g.Gf = y[1] / norm;                             // a^3 E dD1/da
  g.f1 = y[1] / (a * a * g.E * y[0]);             // dlnD1/dlna = G1/(a^2 E D1)
  g.f2 = y[3] / (a * a * g.E * y[2]);
  g.gf = 1.5 * om * g.D1 / (a * a * g.E);         // dGf/da by the growth ODE
  return g;
}

// ------------------------------------------------------------------------------------------
// R2  FFT.  Forward: sum_x rho(x) exp(-2 pi i n.x/ng), unnormalised; inverse: sign +, 1/ng^3.
// 1-D transform: naive O(n^2) DFT for n <= 8, iterative radix-2 otherwise (BASELINE.json
// north_star: "a naive DFT on tiny grids and a simple FFT otherwise").
// ------------------------------------------------------------------------------------------
void dft_naive_1d(cd* a, int n, int sign) {
  std::vector<cd> out(n);
  for (int k = 0; k < n; ++k) {
    cd s(0.0, 0.0);
    for (int j = 0; j < n; ++j) {
      const double ang = sign * 2.0 * PI * (double)((int64_t)j * k % n) / n;
      s += a[j] * cd(std::cos(ang), std::sin(ang));
    }
    out[k] = s;
  }
  for (int k = 0; k < n; ++k) a[k] = out[k];
}

void fft_radix2_1d(cd* a, int n, int sign) {
  // bit reversal
  for (int i = 1, j = 0; i < n; ++i) {
    int bit = n >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) std::swap(a[i], a[j]);
  }
  for (int len = 2; len <= n; len <<= 1) {
    for (int i = 0; i < n; i += len) {
      for (int j = 0; j < len / 2; ++j) {
        const double ang = sign * 2.0 * PI * j / len;
        const cd w(std::cos(ang), std::sin(ang));
        const cd u = a[i + j], v = a[i + j + len / 2] * w;
        a[i + j] = u + v;
        a[i + j + len / 2] = u - v;
      }
    }
  }
}

void fft_1d(cd* a, int n, int sign, bool force_naive) {
  if (n <= 8 || force_naive) dft_naive_1d(a, n, sign);
  else fft_radix2_1d(a, n, sign);
}

// full complex 3-D transform, one axis at a time
void fft3d_complex(std::vector<cd>& a, int ng, int sign, bool force_naive) {
  const int64_t n = ng;
  // z axis (contiguous)
#pragma omp parallel for schedule(static)
  for (int64_t xy = 0; xy < n * n; ++xy) fft_1d(&a[xy * n], ng, sign, force_naive);
  // y axis
#pragma omp parallel
  {
    std::vector<cd> pencil(ng);
#pragma omp for schedule(static)
    for (int64_t xz = 0; xz < n * n; ++xz) {
      const int64_t x = xz / n, z = xz % n;
      for (int64_t y = 0; y < n; ++y) pencil[y] = a[(x * n + y) * n + z];
      fft_1d(pencil.data(), ng, sign, force_naive);
      for (int64_t y = 0; y < n; ++y) a[(x * n + y) * n + z] = pencil[y];
    }
  }
  // x axis
#pragma omp parallel
  {
    std::vector<cd> pencil(ng);
#pragma omp for schedule(static)
    for (int64_t yz = 0; yz < n * n; ++yz) {
      for (int64_t x = 0; x < n; ++x) pencil[x] = a[x * n * n + yz];
      fft_1d(pencil.data(), ng, sign, force_naive);
      for (int64_t x = 0; x < n; ++x) a[x * n * n + yz] = pencil[x];
    }
  }
}

void r2c_impl(const double* real, int ng, double* cplx, bool force_naive) {
  const int64_t n = ng, nzh = ng / 2 + 1;
  std::vector<cd> a(n * n * n);
  for (int64_t i = 0; i < n * n * n; ++i) a[i] = cd(real[i], 0.0);
  fft3d_complex(a, ng, -1, force_naive);
  for (int64_t xy = 0; xy < n * n; ++xy)
    for (int64_t z = 0; z < nzh; ++z) {
      cplx[2 * (xy * nzh + z)] = a[xy * n + z].real();
      cplx[2 * (xy * nzh + z) + 1] = a[xy * n + z].imag();
    }
}

void c2r_impl(const double* cplx, int ng, double* real, bool force_naive) {
  const int64_t n = ng, nzh = ng / 2 + 1;
  std::vector<cd> a(n * n * n);
  // fill the full spectrum from the stored half by Hermitian symmetry a(-k) = conj(a(k))
  for (int64_t x = 0; x < n; ++x)
    for (int64_t y = 0; y < n; ++y)
      for (int64_t z = 0; z < n; ++z) {
        if (z < nzh) {
          const int64_t i = (x * n + y) * nzh + z;
          a[(x * n + y) * n + z] = cd(cplx[2 * i], cplx[2 * i + 1]);
        } else {
          const int64_t xm = (n - x) % n, ym = (n - y) % n, zm = n - z;
          const int64_t i = (xm * n + ym) * nzh + zm;
          a[(x * n + y) * n + z] = cd(cplx[2 * i], -cplx[2 * i + 1]);
        }
      }
  fft3d_complex(a, ng, +1, force_naive);
  const double inv = 1.0 / ((double)n * n * n);
  for (int64_t i = 0; i < n * n * n; ++i) real[i] = a[i].real() * inv;
}

// ------------------------------------------------------------------------------------------
// R1 / R10  Cloud-in-cell window: linear window of unit size; readout uses the
// same kernel.  i_d = floor(x_d), t_d = x_d - i_d, 8 cells (i_d + {0,1}) mod ng.
// ------------------------------------------------------------------------------------------
struct Cic {
  int64_t i0[3], i1[3];
  double t[3];
};

inline Cic cic_of(double x, double y, double z, int64_t ng) {
  Cic c;
  const double p[3] = {x, y, z};
  for (int d = 0; d < 3; ++d) {
    const double fl = std::floor(p[d]);
    c.t[d] = p[d] - fl;
    c.i0[d] = wrap_index((int64_t)fl, ng);
    c.i1[d] = wrap_index((int64_t)fl + 1, ng);
  }
  return c;
}

void paint_impl(const double* pos, const double* mass, double mass_const, int64_t n, int ng,
                double* mesh) {
  const int64_t g = ng;
  std::memset(mesh, 0, sizeof(double) * g * g * g);
  for (int64_t p = 0; p < n; ++p) {
    const Cic c = cic_of(pos[p], pos[n + p], pos[2 * n + p], g);
    const double m = mass ? mass[p] : mass_const;
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 2; ++b)
        for (int e = 0; e < 2; ++e) {
          const double w = (a ? c.t[0] : 1.0 - c.t[0]) * (b ? c.t[1] : 1.0 - c.t[1]) *
                           (e ? c.t[2] : 1.0 - c.t[2]);
          const int64_t ix = a ? c.i1[0] : c.i0[0], iy = b ? c.i1[1] : c.i0[1],
                        iz = e ? c.i1[2] : c.i0[2];
          mesh[(ix * g + iy) * g + iz] += m * w;
        }
  }
}

void readout_impl(const double* mesh, const double* pos, int64_t n, int ng, double* out) {
  const int64_t g = ng;
#pragma omp parallel for schedule(static)
  for (int64_t p = 0; p < n; ++p) {
    const Cic c = cic_of(pos[p], pos[n + p], pos[2 * n + p], g);
    double s = 0.0;
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 2; ++b)
        for (int e = 0; e < 2; ++e) {
          const double w = (a ? c.t[0] : 1.0 - c.t[0]) * (b ? c.t[1] : 1.0 - c.t[1]) *
                           (e ? c.t[2] : 1.0 - c.t[2]);
          const int64_t ix = a ? c.i1[0] : c.i0[0], iy = b ? c.i1[1] : c.i0[1],
                        iz = e ? c.i1[2] : c.i0[2];
          s += mesh[(ix * g + iy) * g + iz] * w;
        }
    out[p] = s;
  }
}

// R11: gradient of the CIC sum with respect to the particle position: the d-th weight factor
// (1-t_d, t_d) is replaced by its derivative (-1, +1).  out_grad[d][p] = sum_c mesh[c] dW/dx_d.
void readout_grad_impl(const double* mesh, const double* pos, int64_t n, int ng, double* out3) {
  const int64_t g = ng;
#pragma omp parallel for schedule(static)
  for (int64_t p = 0; p < n; ++p) {
    const Cic c = cic_of(pos[p], pos[n + p], pos[2 * n + p], g);
    double s[3] = {0, 0, 0};
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 2; ++b)
        for (int e = 0; e < 2; ++e) {
          const double wx = a ? c.t[0] : 1.0 - c.t[0], wy = b ? c.t[1] : 1.0 - c.t[1],
                       wz = e ? c.t[2] : 1.0 - c.t[2];
          const double dx = a ? 1.0 : -1.0, dy = b ? 1.0 : -1.0, dz = e ? 1.0 : -1.0;
          const int64_t ix = a ? c.i1[0] : c.i0[0], iy = b ? c.i1[1] : c.i0[1],
                        iz = e ? c.i1[2] : c.i0[2];
          const double v = mesh[(ix * g + iy) * g + iz];
          s[0] += v * dx * wy * wz;
          s[1] += v * wx * dy * wz;
          s[2] += v * wx * wy * dz;
        }
    out3[p] = s[0];
    out3[n + p] = s[1];
    out3[2 * n + p] = s[2];
  }
}

// ------------------------------------------------------------------------------------------
// R3  Force kernel (Eq. 3-5).
//   mode 0 PAPER : K^2 = sum_d (2 sin(w_d/2))^2  [Eq. 4 read as the 3-point Laplacian symbol],
//                  g(w) = (8 sin w - sin 2w)/6    [Eq. 5]
//   mode 1 NAIVE : K^2 = sum_d w_d^2, g(w) = w    ("the simplest way")
//   mode 2 MIXED : K^2 = sum_d w_d^2, g from Eq. 5
// fhat_d = scale * i g(w_d) deltahat / K^2 ;  1/K^2 := 0 at k = 0 ; g := 0 at n_d = ng/2.
// ------------------------------------------------------------------------------------------
inline int freq_of(int64_t i, int64_t ng) { return (int)(i <= ng / 2 ? i : i - ng); }  // (-ng/2, ng/2]

inline double lap_1d(int mode, double w) {
  if (mode == 0) { const double s = 2.0 * std::sin(0.5 * w); return s * s; }
  return w * w;
}
inline double grad_1d(int mode, double w, bool nyquist) {
  if (nyquist) return 0.0;
  if (mode == 1) return w;
  return (8.0 * std::sin(w) - std::sin(2.0 * w)) / 6.0;
}

void force_kernel_impl(const double* dk, int ng, int mode, double scale, double* fk[3]) {
  const int64_t n = ng, nzh = ng / 2 + 1;
#pragma omp parallel for schedule(static)
  for (int64_t x = 0; x < n; ++x)
    for (int64_t y = 0; y < n; ++y)
      for (int64_t z = 0; z < nzh; ++z) {
        const int64_t idx[3] = {x, y, z};
        double w[3], k2 = 0.0;
        bool nyq[3];
        for (int d = 0; d < 3; ++d) {
          const int f = freq_of(idx[d], n);
          w[d] = 2.0 * PI * f / n;
          nyq[d] = (2 * f == n);
          k2 += lap_1d(mode, w[d]);
        }
        const bool zero = (x == 0 && y == 0 && z == 0);
        const double inv = zero ? 0.0 : 1.0 / k2;
        const int64_t i = (x * n + y) * nzh + z;
        const cd delta(dk[2 * i], dk[2 * i + 1]);
        for (int d = 0; d < 3; ++d) {
          const cd f = cd(0.0, scale * grad_1d(mode, w[d], nyq[d]) * inv) * delta;
          fk[d][2 * i] = f.real();
          fk[d][2 * i + 1] = f.imag();
        }
      }
}

// Alg. 3 ForceGrids(G, mode=local): FFT3D -> grad_i laplace^-1 -> iFFT3D x3.
void force_grids_impl(const double* rho, int ng, int mode, double scale, double* F[3]) {
  const int64_t nk = (int64_t)ng * ng * (ng / 2 + 1);
  std::vector<double> dk(2 * nk), fx(2 * nk), fy(2 * nk), fz(2 * nk);
  r2c_impl(rho, ng, dk.data(), false);
  double* fk[3] = {fx.data(), fy.data(), fz.data()};
  force_kernel_impl(dk.data(), ng, mode, scale, fk);
  for (int d = 0; d < 3; ++d) c2r_impl(fk[d], ng, F[d], false);
}

// ------------------------------------------------------------------------------------------
// N3  Multi-grid pyramid (Eq. 6-9; Alg. 2-3).  DESIGN.md reading R14:
//   * BSpline(6): the paper names "a 3-D bspline kernel of order 6" and nothing else.  Taken as the two-scale
//     (refinement) mask of the order-6 cardinal B-spline, h = [1, 6, 15, 20, 15, 6, 1] / 64 per axis, offsets
//     -3..3, K = h (x) h (x) h, sum 1: the low-pass for which upsampling by EXPAND is exact B-spline
//     subdivision, and the one whose transposed filter needs the paper's factor 8 = 2^3 to interpolate
//     (each polyphase of 2 h sums to 1).
//   * Conv3D(D, K, S = 2), periodic:        out[X] = sum_j K[j] in[(2 X + j) mod n]            (n -> n/2)
//   * TransposedConv3D(H, 8 K, S = 2):      out[x] = sum_X 8 K[x - 2 X] in[X]  (periodic)     (n/2 -> n)
//   * REDUCE / EXPAND apply them f times (Alg. 2: "consecutively f times").
//   * Force (Alg. 3): F = EXPAND(2^f ForceGrids(REDUCE(H))) + F_S - EXPAND(REDUCE(F_S)), F_S = ForceGrids(H).
//     The factor 2^f is units: ForceGrids on the coarse mesh gives the force per COARSE cell spacing
//     (laplace^-1 ~ spacing^2, grad ~ 1/spacing), and one coarse spacing is 2^f fine cells; Alg. 3 is silent.
// Plain loops over the definition; nothing separable, nothing cached.
// ------------------------------------------------------------------------------------------
const double kBspline6[7] = {1.0 / 64, 6.0 / 64, 15.0 / 64, 20.0 / 64, 15.0 / 64, 6.0 / 64, 1.0 / 64};

// one level: in [n^3] -> out [(n/2)^3]
void conv3d_stride2(const double* in, int n, double* out) {
  const int64_t m = n / 2, g = n;
#pragma omp parallel for schedule(static)
  for (int64_t X = 0; X < m; ++X)
    for (int64_t Y = 0; Y < m; ++Y)
      for (int64_t Z = 0; Z < m; ++Z) {
        double s = 0.0;
        for (int a = -3; a <= 3; ++a)
          for (int b = -3; b <= 3; ++b)
            for (int c = -3; c <= 3; ++c) {
              const int64_t x = wrap_index(2 * X + a, g), y = wrap_index(2 * Y + b, g), z = wrap_index(2 * Z + c, g);
              s += kBspline6[a + 3] * kBspline6[b + 3] * kBspline6[c + 3] * in[(x * g + y) * g + z];
            }
        out[(X * m + Y) * m + Z] = s;
      }
}

// one level: in [m^3] -> out [(2m)^3], kernel 8 K
void transposed_conv3d_stride2(const double* in, int m_, double* out) {
  const int64_t m = m_, g = 2 * m;
  std::memset(out, 0, sizeof(double) * g * g * g);
  // scatter form of the definition: coarse cell X contributes 8 K[j] in[X] to fine cell 2 X + j
  for (int64_t X = 0; X < m; ++X)
    for (int64_t Y = 0; Y < m; ++Y)
      for (int64_t Z = 0; Z < m; ++Z) {
        const double v = 8.0 * in[(X * m + Y) * m + Z];
        for (int a = -3; a <= 3; ++a)
          for (int b = -3; b <= 3; ++b)
            for (int c = -3; c <= 3; ++c) {
              const int64_t x = wrap_index(2 * X + a, g), y = wrap_index(2 * Y + b, g), z = wrap_index(2 * Z + c, g);
              out[(x * g + y) * g + z] += kBspline6[a + 3] * kBspline6[b + 3] * kBspline6[c + 3] * v;
            }
      }
}

// Alg. 2 REDUCE(H, f): in [n^3] -> out [(n / 2^f)^3]
void reduce_impl(const double* in, int n, int f, double* out) {
  std::vector<double> cur(in, in + (int64_t)n * n * n), nxt;
  for (int i = 0; i < f; ++i) {
    const int64_t m = n / 2;
    nxt.assign(m * m * m, 0.0);
    conv3d_stride2(cur.data(), n, nxt.data());
    cur.swap(nxt);
    n = (int)m;
  }
  std::memcpy(out, cur.data(), sizeof(double) * cur.size());
}

// Alg. 2 EXPAND(D, f): in [m^3] -> out [(m 2^f)^3]
void expand_impl(const double* in, int m, int f, double* out) {
  std::vector<double> cur(in, in + (int64_t)m * m * m), nxt;
  for (int i = 0; i < f; ++i) {
    const int64_t g = 2 * (int64_t)m;
    nxt.assign(g * g * g, 0.0);
    transposed_conv3d_stride2(cur.data(), m, nxt.data());
    cur.swap(nxt);
    m = (int)g;
  }
  std::memcpy(out, cur.data(), sizeof(double) * cur.size());
}

// Alg. 3 Force(H, f): the three force meshes of the two-level pyramid scheme, in the paper's order
void force_grids_pyramid_impl(const double* rho, int ng, int mode, double scale, int f, double* F[3]) {
  const int nc = ng >> f;
  const int64_t g3 = (int64_t)ng * ng * ng, c3 = (int64_t)nc * nc * nc;
  std::vector<double> D(c3);
  reduce_impl(rho, ng, f, D.data());                                   // D <= REDUCE(H)
  std::vector<double> FL0(c3), FL1(c3), FL2(c3);
  double* FL[3] = {FL0.data(), FL1.data(), FL2.data()};
  force_grids_impl(D.data(), nc, mode, scale * (double)(1 << f), FL);  // F_L <= ForceGrids(D), in fine-cell units
  force_grids_impl(rho, ng, mode, scale, F);                           // F_S <= ForceGrids(H)
  std::vector<double> up(g3), low(c3), lowup(g3);
  for (int d = 0; d < 3; ++d) {
    expand_impl(FL[d], nc, f, up.data());                              // F_iL <= EXPAND(F_iL)
    reduce_impl(F[d], ng, f, low.data());                              // F_il <= REDUCE(F_iS)
    expand_impl(low.data(), nc, f, lowup.data());                      // F_il <= EXPAND(F_il)
    for (int64_t i = 0; i < g3; ++i) F[d][i] = up[i] + (F[d][i] - lowup[i]);   // F_i <= F_iL + (F_iS - F_il)
  }
}

// paint -> ForceGrids -> readout x3 : one force evaluation at the particles.
void force_impl(const double* pos, int64_t n, int ng, int mode, double scale, double mass,
                double* force, double* rho_out) {
  const int64_t g3 = (int64_t)ng * ng * ng;
  std::vector<double> rho(g3), F0(g3), F1(g3), F2(g3);
  paint_impl(pos, nullptr, mass, n, ng, rho.data());
  if (rho_out) std::memcpy(rho_out, rho.data(), sizeof(double) * g3);
  double* F[3] = {F0.data(), F1.data(), F2.data()};
  force_grids_impl(rho.data(), ng, mode, scale, F);
  for (int d = 0; d < 3; ++d) readout_impl(F[d], pos, n, ng, force + d * n);
}

// ------------------------------------------------------------------------------------------
// R4  Kick / drift factors (Eq. 1-2; growth-factor form re-derived by demanding
// a Zel'dovich flow x = q + D1(a) psi be reproduced exactly; mode 1 = plain Quinn et al. integrals).
//   Drift = [D1(af) - D1(ai)] / [ac^3 E(ac) D1'(ac)] = [D1(af) - D1(ai)] / Gf(ac)
//   Kick  = [Gf(af) - Gf(ai)] / [ac^2 E(ac) gf(ac)]
// ------------------------------------------------------------------------------------------
double quinn_integral(double om, double ai, double af, int power) {
  // int_ai^af da / (a^power E(a)) by composite Simpson
  const int m = 2000;
  const double h = (af - ai) / m;
  double s = 0.0;
  for (int i = 0; i <= m; ++i) {
    const double a = ai + i * h;
    const double v = 1.0 / (std::pow(a, power) * E_of_a(om, a));
    s += v * ((i == 0 || i == m) ? 1.0 : (i % 2 ? 4.0 : 2.0));
  }
  return s * h / 3.0;
}

double drift_factor(double om, double ai, double ac, double af, int mode) {
  if (mode == 1) return quinn_integral(om, ai, af, 3);
  const Growth gi = growth_at(om, ai), gc = growth_at(om, ac), gf = growth_at(om, af);
  return (gf.D1 - gi.D1) / gc.Gf;
}
double kick_factor(double om, double ai, double ac, double af, int mode) {
  if (mode == 1) return quinn_integral(om, ai, af, 2);
  const Growth gi = growth_at(om, ai), gc = growth_at(om, ac), gf = growth_at(om, af);
  return (gf.Gf - gi.Gf) / (ac * ac * gc.E * gc.gf);
}

void kick_impl(double* mom, const double* force, int64_t n, double fac) {
  for (int64_t i = 0; i < 3 * n; ++i) mom[i] += force[i] * fac;   // Eq. 2
}
void drift_impl(double* pos, const double* mom, int64_t n, double fac, int ng) {
  for (int64_t i = 0; i < 3 * n; ++i) {                            // Eq. 1, then periodic wrap
    double x = pos[i] + mom[i] * fac;
    x -= ng * std::floor(x / ng);
    if (x >= ng) x -= ng;
    pos[i] = x;
  }
}

// ------------------------------------------------------------------------------------------
// R9  LPT initial conditions (Alg. 4) with spectral kernels on the Np grid.
// ------------------------------------------------------------------------------------------
inline double kcomp(int64_t i, int64_t n, bool zero_nyquist) {
  const int f = freq_of(i, n);
  if (zero_nyquist && 2 * f == n) return 0.0;
  return 2.0 * PI * f / n;
}

// out = c2r( mult(k) * in ), mult = (i k_a)^[a>=0] (i k_b)^[b>=0] * (-1/k^2)^[inv_lap]
// i k_d is zeroed at the Nyquist index of axis d; for a == b the product -(k_a)^2 keeps Nyquist.
void spectral_apply(const std::vector<double>& in_k, int np, int a, int b, bool inv_lap,
                    std::vector<double>& out_real, bool conj_mult = false) {
  const int64_t n = np, nzh = np / 2 + 1;
  std::vector<double> tmp(in_k.size());
#pragma omp parallel for schedule(static)
  for (int64_t x = 0; x < n; ++x)
    for (int64_t y = 0; y < n; ++y)
      for (int64_t z = 0; z < nzh; ++z) {
        const int64_t idx[3] = {x, y, z};
        const int64_t i = (x * n + y) * nzh + z;
        cd m(1.0, 0.0);
        if (a >= 0 && a == b) {
          const double k = kcomp(idx[a], n, false);
          m *= cd(-k * k, 0.0);
        } else {
          if (a >= 0) m *= cd(0.0, kcomp(idx[a], n, true));
          if (b >= 0) m *= cd(0.0, kcomp(idx[b], n, true));
        }
        if (inv_lap) {
          double k2 = 0.0;
          for (int d = 0; d < 3; ++d) { const double k = kcomp(idx[d], n, false); k2 += k * k; }
          m *= (x == 0 && y == 0 && z == 0) ? 0.0 : -1.0 / k2;
        }
        if (conj_mult) m = std::conj(m);   // transpose of a real convolution (R12)
        const cd v = m * cd(in_k[2 * i], in_k[2 * i + 1]);
        tmp[2 * i] = v.real();
        tmp[2 * i + 1] = v.imag();
      }
  out_real.resize(n * n * n);
  c2r_impl(tmp.data(), np, out_real.data(), false);
}

// psi1[3][np^3], psi2[3][np^3] in Np-grid cells (psi2 untouched when order == 1)
void lpt_displacements(const double* delta_lin, int np, int order, std::vector<double> psi1[3],
                       std::vector<double> psi2[3]) {
  const int64_t n3 = (int64_t)np * np * np, nk = (int64_t)np * np * (np / 2 + 1);
  std::vector<double> dk(2 * nk);
  r2c_impl(delta_lin, np, dk.data(), false);
  // psi1_d = c2r( i k_d delta / k^2 ) = c2r( (i k_d) (-1/k^2) (-delta) ): phi1 = -delta/k^2, psi1 = -grad phi1
  std::vector<double> mdk(2 * nk);
  for (int64_t i = 0; i < 2 * nk; ++i) mdk[i] = -dk[i];
  for (int d = 0; d < 3; ++d) spectral_apply(mdk, np, d, -1, true, psi1[d]);
  if (order < 2) return;
  // phi1_,ij = c2r( (i k_i)(i k_j) phihat1 ), phihat1 = -delta/k^2
  std::vector<double> pxx, pyy, pzz, pxy, pxz, pyz;
  spectral_apply(dk, np, 0, 0, true, pxx);
  spectral_apply(dk, np, 1, 1, true, pyy);
  spectral_apply(dk, np, 2, 2, true, pzz);
  spectral_apply(dk, np, 0, 1, true, pxy);
  spectral_apply(dk, np, 0, 2, true, pxz);
  spectral_apply(dk, np, 1, 2, true, pyz);
  std::vector<double> S(n3);
  for (int64_t i = 0; i < n3; ++i)
    S[i] = pxx[i] * pyy[i] + pxx[i] * pzz[i] + pyy[i] * pzz[i] - pxy[i] * pxy[i] -
           pxz[i] * pxz[i] - pyz[i] * pyz[i];
  std::vector<double> Sk(2 * nk);
  r2c_impl(S.data(), np, Sk.data(), false);
  // psi2_d = c2r( -i k_d S / k^2 ) = c2r( (i k_d)(-1/k^2) S ) = grad phi2, lap phi2 = S
  for (int d = 0; d < 3; ++d) spectral_apply(Sk, np, d, -1, true, psi2[d]);
}

void lpt_init_impl(const double* delta_lin, int np, int ng, double om, double a0, int order,
                   double* pos, double* mom) {
  const int64_t n3 = (int64_t)np * np * np;
  const int B = ng / np;
  std::vector<double> psi1[3], psi2[3];
  lpt_displacements(delta_lin, np, order, psi1, psi2);
  const Growth g = growth_at(om, a0);
  const double pre = a0 * a0 * g.E;
  for (int64_t i = 0; i < n3; ++i) {
    const int64_t q[3] = {i / ((int64_t)np * np), (i / np) % np, i % np};
    for (int d = 0; d < 3; ++d) {
      double dx = g.D1 * psi1[d][i];
      double v = pre * g.f1 * g.D1 * psi1[d][i];
      if (order >= 2) {
        dx += g.D2 * psi2[d][i];
        v += pre * g.f2 * g.D2 * psi2[d][i];
      }
      double x = (double)(q[d] * B) + dx * B;    // mesh cells
      x -= ng * std::floor(x / ng);
      if (x >= ng) x -= ng;
      pos[d * n3 + i] = x;
      mom[d * n3 + i] = v * B;
    }
  }
}

// ------------------------------------------------------------------------------------------
// R6  Whole run.  stages a_0..a_n; force at a_0; per step j: a_h = sqrt(a_j a_{j+1});
// kick(a_j -> a_h, force epoch a_j); drift(a_j -> a_{j+1}, momentum epoch a_h);
// force at a_{j+1}; kick(a_h -> a_{j+1}, force epoch a_{j+1}).
// ------------------------------------------------------------------------------------------
void nbody_impl(double* pos, double* mom, int64_t n, int ng, int np, double om, int mode,
                int factor_mode, const double* stages, int n_steps, double* traj) {
  const double B = (double)ng / np, mass = B * B * B, scale = 1.5 * om;
  std::vector<double> f(3 * n);
  force_impl(pos, n, ng, mode, scale, mass, f.data(), nullptr);
  if (traj) std::memcpy(traj, pos, sizeof(double) * 3 * n);
  for (int j = 0; j < n_steps; ++j) {
    const double ai = stages[j], af = stages[j + 1], ah = std::sqrt(ai * af);
    kick_impl(mom, f.data(), n, kick_factor(om, ai, ai, ah, factor_mode));
    drift_impl(pos, mom, n, drift_factor(om, ai, ah, af, factor_mode), ng);
    force_impl(pos, n, ng, mode, scale, mass, f.data(), nullptr);
    if (traj) std::memcpy(traj + (int64_t)(j + 1) * 3 * n, pos, sizeof(double) * 3 * n);
    kick_impl(mom, f.data(), n, kick_factor(om, ah, af, af, factor_mode));
  }
}

// ------------------------------------------------------------------------------------------
// R12  Reverse mode ("differentiable with respect to every component").
// Every forward operation above is transposed in reverse order; nothing is merged or simplified.
//   * T = c2r o mult(k) o r2c is a real periodic convolution; its transpose is the convolution
//     whose multiplier is conj(mult) (correlation theorem).
//   * paint^T (w.r.t. the mesh)  = readout ;  readout^T (w.r.t. the mesh) = paint with mass = cotangent;
//     position derivatives by readout_grad_impl (R11).
//   * wrap() has unit derivative.
// ------------------------------------------------------------------------------------------

// rho_bar = sum_d ForceGrids_d^T Fbar_d : r2c, multiply by conj(scale * i g_d / K^2), sum, c2r.
void force_grids_transpose(double* const Fbar[3], int ng, int mode, double scale, double* rho_bar) {
  const int64_t n = ng, nzh = ng / 2 + 1, nk = n * n * nzh;
  std::vector<double> acc(2 * nk, 0.0), fk(2 * nk);
  for (int d = 0; d < 3; ++d) {
    r2c_impl(Fbar[d], ng, fk.data(), false);
#pragma omp parallel for schedule(static)
    for (int64_t x = 0; x < n; ++x)
      for (int64_t y = 0; y < n; ++y)
        for (int64_t z = 0; z < nzh; ++z) {
          const int64_t idx[3] = {x, y, z};
          double k2 = 0.0;
          for (int e = 0; e < 3; ++e) k2 += lap_1d(mode, 2.0 * PI * freq_of(idx[e], n) / n);
          const int f = freq_of(idx[d], n);
          const bool zero = (x == 0 && y == 0 && z == 0);
          const cd mult(0.0, scale * grad_1d(mode, 2.0 * PI * f / n, 2 * f == n) * (zero ? 0.0 : 1.0 / k2));
          const int64_t i = (x * n + y) * nzh + z;
          const cd v = std::conj(mult) * cd(fk[2 * i], fk[2 * i + 1]);
          acc[2 * i] += v.real();
          acc[2 * i + 1] += v.imag();
        }
  }
  c2r_impl(acc.data(), ng, rho_bar, false);
}

// gx[3][n] += J_f(pos)^T v, where f = force_impl(pos) and v[3][n] is the cotangent of the force.
void force_vjp_impl(const double* pos, int64_t n, int ng, int mode, double scale, double mass,
                    const double* v, double* gx) {
  const int64_t g3 = (int64_t)ng * ng * ng;
  std::vector<double> rho(g3), F0(g3), F1(g3), F2(g3), B0(g3), B1(g3), B2(g3), rho_bar(g3), g(3 * n);
  paint_impl(pos, nullptr, mass, n, ng, rho.data());
  double* F[3] = {F0.data(), F1.data(), F2.data()};
  force_grids_impl(rho.data(), ng, mode, scale, F);
  double* Fbar[3] = {B0.data(), B1.data(), B2.data()};
  for (int d = 0; d < 3; ++d) {
    // f_d = readout(F_d, pos):  cotangent of the mesh = paint(pos, mass = v_d);
    //                           cotangent of pos     = v_d * sum_c F_d[c] dW/dx
    paint_impl(pos, v + d * n, 0.0, n, ng, Fbar[d]);
    readout_grad_impl(F[d], pos, n, ng, g.data());
    for (int e = 0; e < 3; ++e)
      for (int64_t p = 0; p < n; ++p) gx[e * n + p] += v[d * n + p] * g[e * n + p];
  }
  force_grids_transpose(Fbar, ng, mode, scale, rho_bar.data());
  // rho = paint(pos, mass): cotangent of pos = mass * sum_c rho_bar[c] dW/dx
  readout_grad_impl(rho_bar.data(), pos, n, ng, g.data());
  for (int64_t i = 0; i < 3 * n; ++i) gx[i] += mass * g[i];
}

// Reverse of nbody_impl.  traj[(n_steps+1)][3][n]: positions at every force evaluation.
// In: gx, gp = dL/d(final pos, final mom).  Out: gx, gp = dL/d(initial pos, initial mom).
void nbody_vjp_impl(const double* traj, int64_t n, int ng, int np, double om, int mode,
                    int factor_mode, const double* stages, int n_steps, double* gx, double* gp) {
  const double B = (double)ng / np, mass = B * B * B, scale = 1.5 * om;
  std::vector<double> v(3 * n);
  for (int j = n_steps - 1; j >= 0; --j) {
    const double ai = stages[j], af = stages[j + 1], ah = std::sqrt(ai * af);
    const double k1 = kick_factor(om, ai, ai, ah, factor_mode);
    const double dr = drift_factor(om, ai, ah, af, factor_mode);
    const double k2 = kick_factor(om, ah, af, af, factor_mode);
    const double* x1 = traj + (int64_t)(j + 1) * 3 * n;
    const double* x0 = traj + (int64_t)j * 3 * n;
    // mom += k2 f(x_{j+1})
    for (int64_t i = 0; i < 3 * n; ++i) v[i] = k2 * gp[i];
    force_vjp_impl(x1, n, ng, mode, scale, mass, v.data(), gx);
    // pos = wrap(pos + dr mom)
    for (int64_t i = 0; i < 3 * n; ++i) gp[i] += dr * gx[i];
    // mom += k1 f(x_j)
    for (int64_t i = 0; i < 3 * n; ++i) v[i] = k1 * gp[i];
    force_vjp_impl(x0, n, ng, mode, scale, mass, v.data(), gx);
  }
}

// Reverse of lpt_init_impl: gdelta[np^3] = dL/d(delta_lin) given gx, gp = dL/d(pos, mom).
void lpt_init_vjp_impl(const double* delta_lin, int np, int ng, double om, double a0, int order,
                       const double* gx, const double* gp, double* gdelta) {
  const int64_t n3 = (int64_t)np * np * np, nk = (int64_t)np * np * (np / 2 + 1);
  const int B = ng / np;
  const Growth g = growth_at(om, a0);
  const double pre = a0 * a0 * g.E;
  std::vector<double> tmp, rk(2 * nk), bar(n3);
  for (int64_t i = 0; i < n3; ++i) gdelta[i] = 0.0;
  // pos = q B + (D1 psi1 + D2 psi2) B ; mom = pre (f1 D1 psi1 + f2 D2 psi2) B
  // psi1_d = T[(i k_d)(-1/k^2)] (-delta)
  for (int d = 0; d < 3; ++d) {
    for (int64_t i = 0; i < n3; ++i)
      bar[i] = B * (g.D1 * gx[d * n3 + i] + pre * g.f1 * g.D1 * gp[d * n3 + i]);
    r2c_impl(bar.data(), np, rk.data(), false);
    spectral_apply(rk, np, d, -1, true, tmp, true);
    for (int64_t i = 0; i < n3; ++i) gdelta[i] -= tmp[i];
  }
  if (order < 2) return;
  // psi2_d = T[(i k_d)(-1/k^2)] S
  std::vector<double> Sbar(n3, 0.0);
  for (int d = 0; d < 3; ++d) {
    for (int64_t i = 0; i < n3; ++i)
      bar[i] = B * (g.D2 * gx[d * n3 + i] + pre * g.f2 * g.D2 * gp[d * n3 + i]);
    r2c_impl(bar.data(), np, rk.data(), false);
    spectral_apply(rk, np, d, -1, true, tmp, true);
    for (int64_t i = 0; i < n3; ++i) Sbar[i] += tmp[i];
  }
  // S = pxx pyy + pxx pzz + pyy pzz - pxy^2 - pxz^2 - pyz^2 ,  p_ij = T[(i k_i)(i k_j)(-1/k^2)] delta
  std::vector<double> dk(2 * nk), phi[6];
  r2c_impl(delta_lin, np, dk.data(), false);
  const int ia[6] = {0, 1, 2, 0, 0, 1}, ib[6] = {0, 1, 2, 1, 2, 2};
  for (int c = 0; c < 6; ++c) spectral_apply(dk, np, ia[c], ib[c], true, phi[c]);
  for (int c = 0; c < 6; ++c) {
    for (int64_t i = 0; i < n3; ++i) {
      double dS;
      if (c == 0) dS = phi[1][i] + phi[2][i];
      else if (c == 1) dS = phi[0][i] + phi[2][i];
      else if (c == 2) dS = phi[0][i] + phi[1][i];
      else dS = -2.0 * phi[c][i];
      bar[i] = Sbar[i] * dS;
    }
    r2c_impl(bar.data(), np, rk.data(), false);
    spectral_apply(rk, np, ia[c], ib[c], true, tmp, true);
    for (int64_t i = 0; i < n3; ++i) gdelta[i] += tmp[i];
  }
}

// ------------------------------------------------------------------------------------------
// N1  MAP reconstruction of the initial field (Eq. 12; Listing 7.1):
//   -log p = sum_c (delta_e - delta_m)^2 / (2 sigma^2) + 1/2 s^dagger S^-1 s,   delta_m = F(s).
// Readings: F(s) = paint(nbody(lpt_init(s))) with mean density 1, so
// delta_e - delta_m = data - rho_m when data is also a mean-1 density; the prior is diagonal in k:
// 1/2 sum over the FULL k-space of |s_k|^2 inv_power[k], s_k the unnormalised DFT of s, inv_power the
// caller's table 1/<|s_k|^2> on the half-complex layout (Listing 7.1: "prior = sum(r2c(var)^2/power)");
// the listing's chisq has no 1/2 -- Eq. 12 is followed.  Gradient of the prior w.r.t. the real field:
// n^3 c2r(inv_power s_k).  Optimiser: Adam (Listing 7.1), textbook update with bias correction.
// ------------------------------------------------------------------------------------------
void recon_loss_grad_impl(const double* s, int np, int ng, double om, int mode, int factor_mode,
                          double a0, int order, const double* stages, int n_steps, const double* data,
                          double sigma, const double* inv_power, double* grad, double* loss2) {
  const int64_t n = (int64_t)np * np * np, g3 = (int64_t)ng * ng * ng, nzh = np / 2 + 1,
                nk = (int64_t)np * np * nzh;
  const double B = (double)ng / np, mass = B * B * B;
  // forward model
  std::vector<double> pos(3 * n), mom(3 * n), traj((size_t)(n_steps + 1) * 3 * n), rho(g3);
  lpt_init_impl(s, np, ng, om, a0, order, pos.data(), mom.data());
  nbody_impl(pos.data(), mom.data(), n, ng, np, om, mode, factor_mode, stages, n_steps, traj.data());
  paint_impl(pos.data(), nullptr, mass, n, ng, rho.data());
  // likelihood term and its cotangent on the mesh
  std::vector<double> gbar(g3);
  double chi2 = 0.0;
  for (int64_t i = 0; i < g3; ++i) {
    const double r = rho[i] - data[i];
    chi2 += r * r;
    gbar[i] = r / (sigma * sigma);
  }
  loss2[0] = 0.5 * chi2 / (sigma * sigma);
  // reverse: paint -> nbody -> lpt_init
  std::vector<double> gx(3 * n), gp(3 * n, 0.0);
  readout_grad_impl(gbar.data(), pos.data(), n, ng, gx.data());
  for (int64_t i = 0; i < 3 * n; ++i) gx[i] *= mass;
  nbody_vjp_impl(traj.data(), n, ng, np, om, mode, factor_mode, stages, n_steps, gx.data(), gp.data());
  lpt_init_vjp_impl(s, np, ng, om, a0, order, gx.data(), gp.data(), grad);
  // prior term
  std::vector<double> sk(2 * nk), gk(2 * nk), gprior(n);
  r2c_impl(s, np, sk.data(), false);
  double prior = 0.0;
  for (int64_t x = 0; x < np; ++x)
    for (int64_t y = 0; y < np; ++y)
      for (int64_t z = 0; z < nzh; ++z) {
        const int64_t i = (x * np + y) * nzh + z;
        const double wt = (z == 0 || 2 * z == np) ? 1.0 : 2.0;      // Hermitian half implied
        prior += wt * inv_power[i] * (sk[2 * i] * sk[2 * i] + sk[2 * i + 1] * sk[2 * i + 1]);
        gk[2 * i] = inv_power[i] * sk[2 * i] * (double)n;
        gk[2 * i + 1] = inv_power[i] * sk[2 * i + 1] * (double)n;
      }
  loss2[1] = 0.5 * prior;
  c2r_impl(gk.data(), np, gprior.data(), false);
  for (int64_t i = 0; i < n; ++i) grad[i] += gprior[i];
}

// Adam (Kingma & Ba), step t >= 1:  m = b1 m + (1-b1) g ; v = b2 v + (1-b2) g^2 ;
// x -= lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps)
void adam_step_impl(double* x, const double* g, double* m, double* v, int64_t n, double lr, double b1,
                    double b2, double eps, int t) {
  const double c1 = 1.0 - std::pow(b1, t), c2 = 1.0 - std::pow(b2, t);
  for (int64_t i = 0; i < n; ++i) {
    m[i] = b1 * m[i] + (1.0 - b1) * g[i];
    v[i] = b2 * v[i] + (1.0 - b2) * g[i] * g[i];
    x[i] -= lr * (m[i] / c1) / (std::sqrt(v[i] / c2) + eps);
  }
}

// ------------------------------------------------------------------------------------------
// R13  Binned power spectrum: |deltahat|^2 V / n_g^2, bins of width k_f centred on integers,
// half-space weights (2 for 0 < nz < ng/2, else 1); cross spectrum for Eq. 10-11.
// ------------------------------------------------------------------------------------------
void power_impl(const double* ma, const double* mb, int ng, double box, double* pk, double* kmean,
                double* nmodes) {
  const int64_t n = ng, nzh = ng / 2 + 1, nk = n * n * nzh;
  const int nb = ng / 2;
  std::vector<double> ak(2 * nk), bk;
  r2c_impl(ma, ng, ak.data(), false);
  if (mb) { bk.resize(2 * nk); r2c_impl(mb, ng, bk.data(), false); }
  for (int b = 0; b < nb; ++b) pk[b] = kmean[b] = nmodes[b] = 0.0;
  const double norm = box * box * box / ((double)n * n * n * (double)n * n * n);
  const double kf = 2.0 * PI / box;
  for (int64_t x = 0; x < n; ++x)
    for (int64_t y = 0; y < n; ++y)
      for (int64_t z = 0; z < nzh; ++z) {
        const double fx = freq_of(x, n), fy = freq_of(y, n), fz = (double)z;
        const double kn = std::sqrt(fx * fx + fy * fy + fz * fz);
        const int b = (int)std::floor(kn + 0.5) - 1;     // bin b centred on (b+1) k_f
        if (b < 0 || b >= nb) continue;
        const double w = (z > 0 && 2 * z < n) ? 2.0 : 1.0;
        const int64_t i = (x * n + y) * nzh + z;
        double p;
        if (mb) p = ak[2 * i] * bk[2 * i] + ak[2 * i + 1] * bk[2 * i + 1];
        else p = ak[2 * i] * ak[2 * i] + ak[2 * i + 1] * ak[2 * i + 1];
        pk[b] += w * p * norm;
        kmean[b] += w * kn * kf;
        nmodes[b] += w;
      }
  for (int b = 0; b < nb; ++b)
    if (nmodes[b] > 0) { pk[b] /= nmodes[b]; kmean[b] /= nmodes[b]; }
}

}  // namespace

// ============================================================================================
// C interface (host pointers only).  Loaded with ctypes from oracle/__init__.py.
// ============================================================================================
extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// out = {D1, f1, D2, f2, E, Gf, gf}
void orc_growth(double om, double a, double* out) {
  const Growth g = growth_at(om, a);
  out[0] = g.D1; out[1] = g.f1; out[2] = g.D2; out[3] = g.f2; out[4] = g.E; out[5] = g.Gf;
  out[6] = g.gf;
}
double orc_drift_factor(double om, double ai, double ac, double af, int factor_mode) {
  return drift_factor(om, ai, ac, af, factor_mode);
}
double orc_kick_factor(double om, double ai, double ac, double af, int factor_mode) {
  return kick_factor(om, ai, ac, af, factor_mode);
}

void orc_fft_r2c(const double* real, int ng, double* cplx, int force_naive) {
  r2c_impl(real, ng, cplx, force_naive != 0);
}
void orc_fft_c2r(const double* cplx, int ng, double* real, int force_naive) {
  c2r_impl(cplx, ng, real, force_naive != 0);
}

void orc_paint(const double* pos, const double* mass, double mass_const, int64_t n, int ng,
               double* mesh) {
  paint_impl(pos, mass, mass_const, n, ng, mesh);
}
void orc_readout(const double* mesh, const double* pos, int64_t n, int ng, double* out) {
  readout_impl(mesh, pos, n, ng, out);
}

void orc_apply_force_kernel(const double* dk, int ng, int mode, double scale, double* fkx,
                            double* fky, double* fkz) {
  double* fk[3] = {fkx, fky, fkz};
  force_kernel_impl(dk, ng, mode, scale, fk);
}
void orc_force_grids(const double* rho, int ng, int mode, double scale, double* Fx, double* Fy,
                     double* Fz) {
  double* F[3] = {Fx, Fy, Fz};
  force_grids_impl(rho, ng, mode, scale, F);
}
void orc_force(const double* pos, int64_t n, int ng, int mode, double scale, double mass,
               double* force, double* rho_out) {
  force_impl(pos, n, ng, mode, scale, mass, force, rho_out);
}

void orc_reduce(const double* in, int n, int f, double* out) { reduce_impl(in, n, f, out); }
void orc_expand(const double* in, int m, int f, double* out) { expand_impl(in, m, f, out); }
void orc_force_grids_pyramid(const double* rho, int ng, int mode, double scale, int f, double* Fx, double* Fy,
                             double* Fz) {
  double* F[3] = {Fx, Fy, Fz};
  force_grids_pyramid_impl(rho, ng, mode, scale, f, F);
}
// one pyramid force evaluation at the particles: paint -> Alg. 3 Force -> readout x3
void orc_force_pyramid(const double* pos, int64_t n, int ng, int mode, double scale, double mass, int f,
                       double* force) {
  const int64_t g3 = (int64_t)ng * ng * ng;
  std::vector<double> rho(g3), F0(g3), F1(g3), F2(g3);
  paint_impl(pos, nullptr, mass, n, ng, rho.data());
  double* F[3] = {F0.data(), F1.data(), F2.data()};
  force_grids_pyramid_impl(rho.data(), ng, mode, scale, f, F);
  for (int d = 0; d < 3; ++d) readout_impl(F[d], pos, n, ng, force + d * n);
}

void orc_kick(double* mom, const double* force, int64_t n, double factor) {
  kick_impl(mom, force, n, factor);
}
void orc_drift(double* pos, const double* mom, int64_t n, double factor, int ng) {
  drift_impl(pos, mom, n, factor, ng);
}

void orc_lpt_displacements(const double* delta_lin, int np, int order, double* psi1, double* psi2) {
  const int64_t n3 = (int64_t)np * np * np;
  std::vector<double> p1[3], p2[3];
  lpt_displacements(delta_lin, np, order, p1, p2);
  for (int d = 0; d < 3; ++d) {
    std::memcpy(psi1 + d * n3, p1[d].data(), sizeof(double) * n3);
    if (order >= 2 && psi2) std::memcpy(psi2 + d * n3, p2[d].data(), sizeof(double) * n3);
  }
}
void orc_lpt_init(const double* delta_lin, int np, int ng, double om, double a0, int order,
                  double* pos, double* mom) {
  lpt_init_impl(delta_lin, np, ng, om, a0, order, pos, mom);
}

void orc_nbody(double* pos, double* mom, int64_t n, int ng, int np, double om, int mode,
               int factor_mode, const double* stages, int n_steps, double* traj) {
  nbody_impl(pos, mom, n, ng, np, om, mode, factor_mode, stages, n_steps, traj);
}

void orc_power(const double* mesh_a, const double* mesh_b, int ng, double box, double* pk,
               double* kmean, double* nmodes) {
  power_impl(mesh_a, mesh_b, ng, box, pk, kmean, nmodes);
}

// ---- R11 adjoints ---------------------------------------------------------------------------
// paint_adjoint: given gbar = dL/drho:  dL/dm_p = readout(gbar, x)_p ;
//                dL/dx_{p,d} = m_p sum_c gbar[c] dW/dx_d.
void orc_paint_adjoint(const double* pos, const double* mass, double mass_const, int64_t n, int ng,
                       const double* grad_mesh, double* grad_pos, double* grad_mass) {
  readout_grad_impl(grad_mesh, pos, n, ng, grad_pos);
  for (int d = 0; d < 3; ++d)
    for (int64_t p = 0; p < n; ++p) grad_pos[d * n + p] *= mass ? mass[p] : mass_const;
  if (grad_mass) readout_impl(grad_mesh, pos, n, ng, grad_mass);
}
// readout_adjoint: given vbar_p = dL/dout_p:  dL/dF += paint(x, mass = vbar) ;
//                  dL/dx_{p,d} = vbar_p sum_c F[c] dW/dx_d.
void orc_readout_adjoint(const double* mesh, const double* pos, int64_t n, int ng,
                         const double* grad_out, double* grad_mesh, double* grad_pos) {
  const int64_t g3 = (int64_t)ng * ng * ng;
  std::vector<double> tmp(g3);
  paint_impl(pos, grad_out, 0.0, n, ng, tmp.data());
  for (int64_t i = 0; i < g3; ++i) grad_mesh[i] += tmp[i];
  if (grad_pos) {
    readout_grad_impl(mesh, pos, n, ng, grad_pos);
    for (int d = 0; d < 3; ++d)
      for (int64_t p = 0; p < n; ++p) grad_pos[d * n + p] *= grad_out[p];
  }
}


// ---- R12 reverse mode ---------------------------------------------------------------------------
void orc_force_vjp(const double* pos, int64_t n, int ng, int mode, double scale, double mass,
                   const double* v, double* gx) {
  force_vjp_impl(pos, n, ng, mode, scale, mass, v, gx);
}
void orc_nbody_vjp(const double* traj, int64_t n, int ng, int np, double om, int mode, int factor_mode,
                   const double* stages, int n_steps, double* gx, double* gp) {
  nbody_vjp_impl(traj, n, ng, np, om, mode, factor_mode, stages, n_steps, gx, gp);
}
void orc_lpt_init_vjp(const double* delta_lin, int np, int ng, double om, double a0, int order,
                      const double* gx, const double* gp, double* gdelta) {
  lpt_init_vjp_impl(delta_lin, np, ng, om, a0, order, gx, gp, gdelta);
}


// ---- N1 reconstruction ----------------------------------------------------------------------------
void orc_recon_loss_grad(const double* s, int np, int ng, double om, int mode, int factor_mode, double a0,
                         int order, const double* stages, int n_steps, const double* data, double sigma,
                         const double* inv_power, double* grad, double* loss2) {
  recon_loss_grad_impl(s, np, ng, om, mode, factor_mode, a0, order, stages, n_steps, data, sigma,
                       inv_power, grad, loss2);
}
void orc_adam_step(double* x, const double* g, double* m, double* v, int64_t n, double lr, double b1,
                   double b2, double eps, int t) {
  adam_step_impl(x, g, m, v, n, lr, b1, b2, eps, t);
}

}  // extern "C"
