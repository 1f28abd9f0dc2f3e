// oracle/oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, obviously-correct fp64 CPU implementation of the checkerboard overrelaxation
// sweep for lattice Landau gauge fixing (arXiv:1412.3655, "cuLGT: Lattice Gauge Fixing on
// GPUs"), written from the paper's text.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may call it.  It shares no code with the CUDA path under
// paper_1412_3655_b200/ (no headers, helpers, tables, pre- or post-processing) and neither
// imports the other.
//
// Citations: P:Lnn = /root/reference/PAPER.md line nn.  "C-n" = reading n in DESIGN.md
// (points where the paper is silent / ambiguous).
//
// Layout (canonical): site s = x0 + N0*(x1 + N1*(x2 + N2*x3)), periodic,
// parity(x) = (x0+x1+x2+x3)&1, black = 0 (C-1).  U is double[V][4][nc][nc][2], i.e. full
// nc x nc complex matrices, re/im interleaved, row-major.  nc = 2 or 3.
//
// There is no blocking, fusion or reordering: every function is the paper's formula looped
// over sites.  Sums over the lattice are Neumaier-compensated so the oracle is the trustworthy
// side of a reduction comparison.  OpenMP is used only across the independent sites of one
// parity ("only transformations at neighboring sites interfere") and across sites in the
// per-site terms of a reduction; the arithmetic per site is unchanged by it.
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"): see DESIGN.md "Oracle pins".
// Every exported function below is pinned by at least one of them; none is "parity unpinned".

#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;

namespace {

int g_threads = 1;

struct Lat {
  int N[4];
  int64_t V;
  int nc;
};

Lat make_lat(const int32_t* dims, int nc) {
  Lat L;
  for (int i = 0; i < 4; ++i) L.N[i] = dims[i];
  L.V = (int64_t)dims[0] * dims[1] * dims[2] * dims[3];
  L.nc = nc;
  return L;
}

void coords_of(const Lat& L, int64_t s, int x[4]) {
  x[0] = (int)(s % L.N[0]); s /= L.N[0];
  x[1] = (int)(s % L.N[1]); s /= L.N[1];
  x[2] = (int)(s % L.N[2]); s /= L.N[2];
  x[3] = (int)s;
}

int64_t index_of(const Lat& L, const int x[4]) {
  return x[0] + (int64_t)L.N[0] * (x[1] + (int64_t)L.N[1] * (x[2] + (int64_t)L.N[2] * x[3]));
}

// site index of x + step*mu_hat with periodic wrap (C-2)
int64_t neighbour(const Lat& L, int64_t s, int mu, int step) {
  int x[4];
  coords_of(L, s, x);
  x[mu] = ((x[mu] + step) % L.N[mu] + L.N[mu]) % L.N[mu];
  return index_of(L, x);
}

int parity_of(const Lat& L, int64_t s) {
  int x[4];
  coords_of(L, s, x);
  return (x[0] + x[1] + x[2] + x[3]) & 1;
}

struct Mat {
  cd e[3][3];
};

Mat zero_mat() {
  Mat m;
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) m.e[a][b] = cd(0.0, 0.0);
  return m;
}

Mat unit_mat(int nc) {
  Mat m = zero_mat();
  for (int a = 0; a < nc; ++a) m.e[a][a] = cd(1.0, 0.0);
  return m;
}

Mat load_mat(const double* base, int nc) {
  Mat m = zero_mat();
  for (int a = 0; a < nc; ++a)
    for (int b = 0; b < nc; ++b) m.e[a][b] = cd(base[2 * (a * nc + b)], base[2 * (a * nc + b) + 1]);
  return m;
}

void store_mat(double* base, int nc, const Mat& m) {
  for (int a = 0; a < nc; ++a)
    for (int b = 0; b < nc; ++b) {
      base[2 * (a * nc + b)] = m.e[a][b].real();
      base[2 * (a * nc + b) + 1] = m.e[a][b].imag();
    }
}

const double* link_ptr(const double* U, const Lat& L, int64_t s, int mu) {
  return U + ((s * 4 + mu) * L.nc * L.nc) * 2;
}
double* link_ptr(double* U, const Lat& L, int64_t s, int mu) {
  return U + ((s * 4 + mu) * L.nc * L.nc) * 2;
}

Mat mul(const Mat& A, const Mat& B, int nc) {
  Mat C = zero_mat();
  for (int a = 0; a < nc; ++a)
    for (int b = 0; b < nc; ++b) {
      cd acc(0.0, 0.0);
      for (int k = 0; k < nc; ++k) acc += A.e[a][k] * B.e[k][b];
      C.e[a][b] = acc;
    }
  return C;
}

Mat dagger(const Mat& A, int nc) {
  Mat C = zero_mat();
  for (int a = 0; a < nc; ++a)
    for (int b = 0; b < nc; ++b) C.e[a][b] = std::conj(A.e[b][a]);
  return C;
}

Mat add(const Mat& A, const Mat& B, int nc) {
  Mat C = zero_mat();
  for (int a = 0; a < nc; ++a)
    for (int b = 0; b < nc; ++b) C.e[a][b] = A.e[a][b] + B.e[a][b];
  return C;
}

cd trace(const Mat& A, int nc) {
  cd t(0.0, 0.0);
  for (int a = 0; a < nc; ++a) t += A.e[a][a];
  return t;
}

// Neumaier-compensated sum of n doubles, in index order.
double neumaier_sum(const double* v, int64_t n) {
  double sum = 0.0, comp = 0.0;
  for (int64_t i = 0; i < n; ++i) {
    double t = sum + v[i];
    if (std::fabs(sum) >= std::fabs(v[i])) comp += (sum - t) + v[i];
    else comp += (v[i] - t) + sum;
    sum = t;
  }
  return sum + comp;
}

// K(x) = sum_mu [ U_mu(x) + U_mu(x - mu)^dagger ]   -- eq. (3).  mu ascending, up then down (C-17).
Mat gather_K(const double* U, const Lat& L, int64_t s) {
  Mat K = zero_mat();
  for (int mu = 0; mu < 4; ++mu) {
    K = add(K, load_mat(link_ptr(U, L, s, mu), L.nc), L.nc);
    int64_t sd = neighbour(L, s, mu, -1);
    K = add(K, dagger(load_mat(link_ptr(U, L, sd, mu), L.nc), L.nc), L.nc);
  }
  return K;
}

// Exact group power q^omega of a unit quaternion q = (c, v) = cos(alpha) + i sin(alpha) n.sigma on
// the principal branch alpha in [0, pi] (reading C-8 of "replacing g(x) by g^omega(x)").
// alpha = atan2(|v|, c), never acos(c).
void su2_pow(const double q[4], double omega, double out[4]) {
  double c = q[0];
  double r = std::hypot(q[1], q[2], q[3]);
  if (r < 1e-150) {
    if (c > 0.0) { out[0] = 1.0; out[1] = out[2] = out[3] = 0.0; }
    else { out[0] = std::cos(omega * M_PI); out[1] = 0.0; out[2] = 0.0; out[3] = std::sin(omega * M_PI); }
    return;
  }
  double alpha = std::atan2(r, c);
  double f = std::sin(omega * alpha) / r;
  out[0] = std::cos(omega * alpha);
  out[1] = q[1] * f;
  out[2] = q[2] * f;
  out[3] = q[3] * f;
}

// SU(2) convention C-7: (a0,a1,a2,a3) <-> [[a0 + i a3, a2 + i a1], [-a2 + i a1, a0 - i a3]].
// Embeds the quaternion q into rows/cols (i,j) of an nc x nc identity.
Mat embed_su2(const double q[4], int i, int j, int nc) {
  Mat g = unit_mat(nc);
  g.e[i][i] = cd(q[0], q[3]);
  g.e[i][j] = cd(q[2], q[1]);
  g.e[j][i] = cd(-q[2], q[1]);
  g.e[j][j] = cd(q[0], -q[3]);
  return g;
}

// One subgroup step (readings C-6, C-9, C-10): project the (i,j) 2x2 block of K onto
// its real-quaternion part p (twice the SU(2)-proportional part), g = p^dagger/|p| which is
// K_block^dagger / sqrt(det K_block^dagger) for an SU(2)-proportional block, raise it to
// the power omega.  Returns false (g_s = 1) when |p| = 0.
bool subgroup_step(const Mat& K, int i, int j, double omega, int nc, Mat* gs) {
  double p0 = K.e[i][i].real() + K.e[j][j].real();
  double p1 = K.e[i][j].imag() + K.e[j][i].imag();
  double p2 = K.e[i][j].real() - K.e[j][i].real();
  double p3 = K.e[i][i].imag() - K.e[j][j].imag();
  double n = std::sqrt(p0 * p0 + p1 * p1 + p2 * p2 + p3 * p3);
  if (n == 0.0) { *gs = unit_mat(nc); return false; }
  double g[4] = {p0 / n, -p1 / n, -p2 / n, -p3 / n};
  double q[4];
  su2_pow(g, omega, q);
  *gs = embed_su2(q, i, j, nc);
  return true;
}

// The site's gauge transformation G from K(x).  SU(2): one step.  SU(3): the three SU(2)
// subgroups (0,1),(0,2),(1,2) in this order, one pass, each seeing K already rotated by the
// previous ones (C-6), omega applied per subgroup (C-10).
Mat site_G(Mat K, double omega, int nc) {
  Mat G = unit_mat(nc);
  static const int pairs[3][2] = {{0, 1}, {0, 2}, {1, 2}};
  int npairs = (nc == 2) ? 1 : 3;
  for (int t = 0; t < npairs; ++t) {
    Mat gs;
    if (!subgroup_step(K, pairs[t][0], pairs[t][1], omega, nc, &gs)) continue;
    K = mul(gs, K, nc);
    G = mul(gs, G, nc);
  }
  return G;
}

}  // namespace

extern "C" {

// Number of OpenMP threads used across independent sites (1 = serial).  Returns the value set.
int oracle_set_threads(int n) {
#ifdef _OPENMP
  g_threads = n < 1 ? 1 : n;
#else
  (void)n;
  g_threads = 1;
#endif
  return g_threads;
}

int oracle_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void oracle_su2_pow(const double* q, double omega, double* out) { su2_pow(q, omega, out); }

// K(x) for every site: out is double[V][nc][nc][2].  eq. (3).
void oracle_K(const int32_t* dims, int nc, const double* U, double* out) {
  Lat L = make_lat(dims, nc);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) store_mat(out + s * nc * nc * 2, nc, gather_K(U, L, s));
}

// G for a given K (one site): K, G are double[nc][nc][2].  P:L50-54.
void oracle_site_G(int nc, const double* K, double omega, double* G) {
  store_mat(G, nc, site_G(load_mat(K, nc), omega, nc));
}

// One subgroup step on a given K: gs = embedded q^omega, returns 1 if |p| > 0.
int oracle_subgroup_step(int nc, const double* K, int i, int j, double omega, double* gs) {
  Mat g;
  bool ok = subgroup_step(load_mat(K, nc), i, j, omega, nc, &g);
  store_mat(gs, nc, g);
  return ok ? 1 : 0;
}

// One HALF sweep over the sites of `parity`, in place (P:L54 checkerboard; C-12).
//   K = sum_mu U_mu(x) + U_mu(x-mu)^dagger                        eq. (3)
//   G = site_G(K, omega)
//   U_mu(x) <- G U_mu(x);  U_mu(x-mu) <- U_mu(x-mu) G^dagger      P:L19-21 with g = 1 elsewhere
void oracle_or_sweep(const int32_t* dims, int nc, double* U, int parity, double omega) {
  Lat L = make_lat(dims, nc);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) {
    if (parity_of(L, s) != parity) continue;
    Mat G = site_G(gather_K(U, L, s), omega, nc);
    Mat Gd = dagger(G, nc);
    for (int mu = 0; mu < 4; ++mu) {
      double* up = link_ptr(U, L, s, mu);
      store_mat(up, nc, mul(G, load_mat(up, nc), nc));
      double* dn = link_ptr(U, L, neighbour(L, s, mu, -1), mu);
      store_mat(dn, nc, mul(load_mat(dn, nc), Gd, nc));
    }
  }
}

// F^U = 1/(N_d N_c V) sum_x sum_mu Re tr U_mu(x)     eq. (2) at g = 1; N_d = 4.
double oracle_functional(const int32_t* dims, int nc, const double* U) {
  Lat L = make_lat(dims, nc);
  std::vector<double> term(L.V);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) {
    double t = 0.0;
    for (int mu = 0; mu < 4; ++mu) t += trace(load_mat(link_ptr(U, L, s, mu), nc), nc).real();
    term[s] = t;
  }
  return neumaier_sum(term.data(), L.V) / (4.0 * nc * (double)L.V);
}

namespace {
// A_mu(x) = [ (U - U^dagger) / (2i) ]_traceless with a*g = 1 (C-4).   P:L31-33.
Mat gauge_field_A(const Mat& Um, int nc) {
  Mat Ud = dagger(Um, nc);
  Mat A = zero_mat();
  const cd two_i(0.0, 2.0);
  for (int a = 0; a < nc; ++a)
    for (int b = 0; b < nc; ++b) A.e[a][b] = (Um.e[a][b] - Ud.e[a][b]) / two_i;
  cd tr = trace(A, nc) / (double)nc;
  for (int a = 0; a < nc; ++a) A.e[a][a] -= tr;
  return A;
}
// Delta(x) = sum_mu ( A_mu(x) - A_mu(x - mu) )     eq. (1).
Mat delta_at(const double* U, const Lat& L, int64_t s) {
  Mat D = zero_mat();
  for (int mu = 0; mu < 4; ++mu) {
    Mat Ax = gauge_field_A(load_mat(link_ptr(U, L, s, mu), L.nc), L.nc);
    Mat Ad = gauge_field_A(load_mat(link_ptr(U, L, neighbour(L, s, mu, -1), mu), L.nc), L.nc);
    for (int a = 0; a < L.nc; ++a)
      for (int b = 0; b < L.nc; ++b) D.e[a][b] += Ax.e[a][b] - Ad.e[a][b];
  }
  return D;
}
}  // namespace

// Delta(x) for every site: out is double[V][nc][nc][2].
void oracle_delta(const int32_t* dims, int nc, const double* U, double* out) {
  Lat L = make_lat(dims, nc);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) store_mat(out + s * nc * nc * 2, nc, delta_at(U, L, s));
}

// theta = 1/(N_c V) sum_x tr[ Delta(x) Delta(x)^dagger ]   (BASELINE.json north_star; C-5).
double oracle_gauge_precision(const int32_t* dims, int nc, const double* U) {
  Lat L = make_lat(dims, nc);
  std::vector<double> term(L.V);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) {
    Mat D = delta_at(U, L, s);
    term[s] = trace(mul(D, dagger(D, nc), nc), nc).real();
  }
  return neumaier_sum(term.data(), L.V) / ((double)nc * (double)L.V);
}

// U_mu(x) <- g(x) U_mu(x) g(x+mu)^dagger for all x, mu.  g is double[V][nc][nc][2], read-only.
void oracle_gauge_transform(const int32_t* dims, int nc, double* U, const double* g) {
  Lat L = make_lat(dims, nc);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) {
    Mat gx = load_mat(g + s * nc * nc * 2, nc);
    for (int mu = 0; mu < 4; ++mu) {
      Mat gf = load_mat(g + neighbour(L, s, mu, +1) * nc * nc * 2, nc);
      double* p = link_ptr(U, L, s, mu);
      store_mat(p, nc, mul(mul(gx, load_mat(p, nc), nc), dagger(gf, nc), nc));
    }
  }
}

// Average plaquette 1/(6 N_c V) sum_x sum_{mu<nu} Re tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^dagger U_nu(x)^dagger].
// Test-only gauge-invariant observable (not on the hot path).
double oracle_plaquette(const int32_t* dims, int nc, const double* U) {
  Lat L = make_lat(dims, nc);
  std::vector<double> term(L.V);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) {
    double t = 0.0;
    for (int mu = 0; mu < 4; ++mu)
      for (int nu = mu + 1; nu < 4; ++nu) {
        Mat a = load_mat(link_ptr(U, L, s, mu), nc);
        Mat b = load_mat(link_ptr(U, L, neighbour(L, s, mu, +1), nu), nc);
        Mat c = dagger(load_mat(link_ptr(U, L, neighbour(L, s, nu, +1), mu), nc), nc);
        Mat d = dagger(load_mat(link_ptr(U, L, s, nu), nc), nc);
        t += trace(mul(mul(a, b, nc), mul(c, d, nc), nc), nc).real();
      }
    term[s] = t;
  }
  return neumaier_sum(term.data(), L.V) / (6.0 * nc * (double)L.V);
}

// 12-parameter representation: keep rows 0,1 of every SU(3) link, rebuild
// row 2 = conj(row0 x row1) in fp64.  n = number of 3x3 matrices in `M` (double[n][3][3][2]).
// Used to give the oracle exactly the field a 12-parameter store holds.
void oracle_reconstruct12(int64_t n, double* M) {
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t k = 0; k < n; ++k) {
    Mat m = load_mat(M + k * 18, 3);
    m.e[2][0] = std::conj(m.e[0][1] * m.e[1][2] - m.e[0][2] * m.e[1][1]);
    m.e[2][1] = std::conj(m.e[0][2] * m.e[1][0] - m.e[0][0] * m.e[1][2]);
    m.e[2][2] = std::conj(m.e[0][0] * m.e[1][1] - m.e[0][1] * m.e[1][0]);
    store_mat(M + k * 18, 3, m);
  }
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// Coulomb gauge (named by the paper beside Landau gauge, P:L7; its details are in the
// paper's ref. [2], which is not available -- DESIGN.md reading C-22):
// the Landau formulas with mu restricted to the 3 spatial directions, time-slice by time-slice.
//   F_t   = 1/(3 N_c V_s) sum_{x in slice t} sum_{i<3} Re tr U_i(x)                (eq. (2), i < 3)
//   K_C(x) = sum_{i<3} [ U_i(x) + U_i(x-i)^dagger ]                                (eq. (3), i < 3)
//   Delta_C(x) = sum_{i<3} ( A_i(x) - A_i(x-i) ),  theta_t = 1/(N_c V_s) sum_{x in t} tr[Delta_C Delta_C^dagger]
// The site update is the same G = site_G(K_C, omega); being a gauge transformation g(x) it acts
// on ALL 8 links touching x, time links included, although they do not enter K_C.
// ---------------------------------------------------------------------------------------------
namespace {
Mat gather_K_spatial(const double* U, const Lat& L, int64_t s) {
  Mat K = zero_mat();
  for (int mu = 0; mu < 3; ++mu) {
    K = add(K, load_mat(link_ptr(U, L, s, mu), L.nc), L.nc);
    int64_t sd = neighbour(L, s, mu, -1);
    K = add(K, dagger(load_mat(link_ptr(U, L, sd, mu), L.nc), L.nc), L.nc);
  }
  return K;
}
Mat delta_spatial_at(const double* U, const Lat& L, int64_t s) {
  Mat D = zero_mat();
  for (int mu = 0; mu < 3; ++mu) {
    Mat Ax = gauge_field_A(load_mat(link_ptr(U, L, s, mu), L.nc), L.nc);
    Mat Ad = gauge_field_A(load_mat(link_ptr(U, L, neighbour(L, s, mu, -1), mu), L.nc), L.nc);
    for (int a = 0; a < L.nc; ++a)
      for (int b = 0; b < L.nc; ++b) D.e[a][b] += Ax.e[a][b] - Ad.e[a][b];
  }
  return D;
}
}  // namespace

extern "C" {

// K_C(x) for every site: out is double[V][nc][nc][2].
void oracle_K_coulomb(const int32_t* dims, int nc, const double* U, double* out) {
  Lat L = make_lat(dims, nc);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) store_mat(out + s * nc * nc * 2, nc, gather_K_spatial(U, L, s));
}

// Delta_C(x) for every site: out is double[V][nc][nc][2].
void oracle_delta_coulomb(const int32_t* dims, int nc, const double* U, double* out) {
  Lat L = make_lat(dims, nc);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) store_mat(out + s * nc * nc * 2, nc, delta_spatial_at(U, L, s));
}

// One HALF sweep of Coulomb-gauge overrelaxation over the sites of `parity`, in place.
void oracle_or_sweep_coulomb(const int32_t* dims, int nc, double* U, int parity, double omega) {
  Lat L = make_lat(dims, nc);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) {
    if (parity_of(L, s) != parity) continue;
    Mat G = site_G(gather_K_spatial(U, L, s), omega, nc);
    Mat Gd = dagger(G, nc);
    for (int mu = 0; mu < 4; ++mu) {
      double* up = link_ptr(U, L, s, mu);
      store_mat(up, nc, mul(G, load_mat(up, nc), nc));
      double* dn = link_ptr(U, L, neighbour(L, s, mu, -1), mu);
      store_mat(dn, nc, mul(load_mat(dn, nc), Gd, nc));
    }
  }
}

// The same half-sweep restricted to the time-slices with active[t] != 0 (slices decouple, so a
// slice whose theta_t has reached the target can stop while the others go on; SURVEY.md 8(f) NEXT-1
// "each slice its own theta_t and stop").  active is uint8[N3].
void oracle_or_sweep_coulomb_masked(const int32_t* dims, int nc, double* U, int parity, double omega,
                                    const uint8_t* active) {
  Lat L = make_lat(dims, nc);
  const int64_t Vs = (int64_t)L.N[0] * L.N[1] * L.N[2];
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) {
    if (parity_of(L, s) != parity || !active[s / Vs]) continue;
    Mat G = site_G(gather_K_spatial(U, L, s), omega, nc);
    Mat Gd = dagger(G, nc);
    for (int mu = 0; mu < 4; ++mu) {
      double* up = link_ptr(U, L, s, mu);
      store_mat(up, nc, mul(G, load_mat(up, nc), nc));
      double* dn = link_ptr(U, L, neighbour(L, s, mu, -1), mu);
      store_mat(dn, nc, mul(load_mat(dn, nc), Gd, nc));
    }
  }
}

// theta_t and F_t for every time-slice t = x3: both are double[N3].
void oracle_coulomb_theta_F(const int32_t* dims, int nc, const double* U, double* theta_t, double* F_t) {
  Lat L = make_lat(dims, nc);
  const int64_t Vs = (int64_t)L.N[0] * L.N[1] * L.N[2];
  std::vector<double> th(L.V), f(L.V);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) {
    Mat D = delta_spatial_at(U, L, s);
    th[s] = trace(mul(D, dagger(D, nc), nc), nc).real();
    double t = 0.0;
    for (int mu = 0; mu < 3; ++mu) t += trace(load_mat(link_ptr(U, L, s, mu), nc), nc).real();
    f[s] = t;
  }
  for (int t = 0; t < L.N[3]; ++t) {          // sites of slice t are contiguous in canonical order
    theta_t[t] = neumaier_sum(th.data() + t * Vs, Vs) / ((double)nc * (double)Vs);
    F_t[t] = neumaier_sum(f.data() + t * Vs, Vs) / (3.0 * nc * (double)Vs);
  }
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// Re-unitarisation (reading C-13/C-23; SURVEY.md 8(f) NEXT-2c).  Not part of the paper's
// text: long fp32 runs let the stored rows drift off the group (C-13), and the projection back is
// the Gram-Schmidt step the 12-parameter representation already implies (the third
// row IS conj(row0 x row1)):  r0 <- r0/|r0|;  r1 <- r1 - <r0,r1> r0;  r1 <- r1/|r1|;
// r2 <- conj(r0 x r1),  <a,b> = sum_k conj(a_k) b_k.   SU(2): (a0..a3) <- (a0..a3)/|a|, applied
// to the first row of the 2x2 matrix and the second row rebuilt as (-conj(b), conj(a)).
// ---------------------------------------------------------------------------------------------
extern "C" {

// n matrices, M = double[n][nc][nc][2], in place.
void oracle_reunitarize(int64_t n, int nc, double* M) {
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t k = 0; k < n; ++k) {
    Mat m = load_mat(M + k * nc * nc * 2, nc);
    if (nc == 2) {
      double nrm = std::sqrt(std::norm(m.e[0][0]) + std::norm(m.e[0][1]));
      cd a = m.e[0][0] / nrm, b = m.e[0][1] / nrm;
      m.e[0][0] = a;  m.e[0][1] = b;
      m.e[1][0] = -std::conj(b);  m.e[1][1] = std::conj(a);
    } else {
      double n0 = 0.0;
      for (int c = 0; c < 3; ++c) n0 += std::norm(m.e[0][c]);
      n0 = std::sqrt(n0);
      for (int c = 0; c < 3; ++c) m.e[0][c] /= n0;
      cd ip(0.0, 0.0);
      for (int c = 0; c < 3; ++c) ip += std::conj(m.e[0][c]) * m.e[1][c];
      for (int c = 0; c < 3; ++c) m.e[1][c] -= ip * m.e[0][c];
      double n1 = 0.0;
      for (int c = 0; c < 3; ++c) n1 += std::norm(m.e[1][c]);
      n1 = std::sqrt(n1);
      for (int c = 0; c < 3; ++c) m.e[1][c] /= n1;
      m.e[2][0] = std::conj(m.e[0][1] * m.e[1][2] - m.e[0][2] * m.e[1][1]);
      m.e[2][1] = std::conj(m.e[0][2] * m.e[1][0] - m.e[0][0] * m.e[1][2]);
      m.e[2][2] = std::conj(m.e[0][0] * m.e[1][1] - m.e[0][1] * m.e[1][0]);
    }
    store_mat(M + k * nc * nc * 2, nc, m);
  }
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// Truncated-series overrelaxation (reading C-24; SURVEY.md 8(f) NEXT-2b).  The paper
// only says "replacing g(x) by g^omega(x)" (citing Mandula-Ogilvie); reading C-8 takes the
// exact power.  This selectable variant takes the binomial series instead,
//     g^omega ~ S_N = sum_{n=0}^{N} binom(omega, n) (g - 1)^n ,
// truncated after order N and projected back to SU(2) by dividing by sqrt(det S_N) (S_N is a
// complex polynomial in g, hence of the form a + i b n.sigma with det = a^2 + b^2).  Everything is
// written out literally with 2x2 complex matrices.  The rest of the update is unchanged.
// ---------------------------------------------------------------------------------------------
namespace {
void su2_pow_series(const double q[4], double omega, int order, double out[4]) {
  Mat g = embed_su2(q, 0, 1, 2);
  Mat m = add(g, unit_mat(2), 2);                       // m = g - 1
  m.e[0][0] -= cd(2.0, 0.0);
  m.e[1][1] -= cd(2.0, 0.0);
  Mat term = unit_mat(2);                               // binom(omega, n) (g-1)^n, n = 0
  Mat sum = unit_mat(2);
  for (int n = 1; n <= order; ++n) {
    term = mul(term, m, 2);
    double ratio = (omega - (double)(n - 1)) / (double)n;   // binom(w,n) = binom(w,n-1) (w-n+1)/n
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 2; ++b) term.e[a][b] *= ratio;
    sum = add(sum, term, 2);
  }
  cd det = sum.e[0][0] * sum.e[1][1] - sum.e[0][1] * sum.e[1][0];
  double nrm = std::sqrt(det.real());
  // back to (a0,a1,a2,a3): [[a0 + i a3, a2 + i a1], ...]   (C-7)
  out[0] = sum.e[0][0].real() / nrm;
  out[3] = sum.e[0][0].imag() / nrm;
  out[2] = sum.e[0][1].real() / nrm;
  out[1] = sum.e[0][1].imag() / nrm;
}

bool subgroup_step_series(const Mat& K, int i, int j, double omega, int order, int nc, Mat* gs) {
  double p0 = K.e[i][i].real() + K.e[j][j].real();
  double p1 = K.e[i][j].imag() + K.e[j][i].imag();
  double p2 = K.e[i][j].real() - K.e[j][i].real();
  double p3 = K.e[i][i].imag() - K.e[j][j].imag();
  double n = std::sqrt(p0 * p0 + p1 * p1 + p2 * p2 + p3 * p3);
  if (n == 0.0) { *gs = unit_mat(nc); return false; }
  double g[4] = {p0 / n, -p1 / n, -p2 / n, -p3 / n};
  double q[4];
  su2_pow_series(g, omega, order, q);
  *gs = embed_su2(q, i, j, nc);
  return true;
}

Mat site_G_series(Mat K, double omega, int order, int nc) {
  Mat G = unit_mat(nc);
  static const int pairs[3][2] = {{0, 1}, {0, 2}, {1, 2}};
  int npairs = (nc == 2) ? 1 : 3;
  for (int t = 0; t < npairs; ++t) {
    Mat gs;
    if (!subgroup_step_series(K, pairs[t][0], pairs[t][1], omega, order, nc, &gs)) continue;
    K = mul(gs, K, nc);
    G = mul(gs, G, nc);
  }
  return G;
}
}  // namespace

extern "C" {

void oracle_su2_pow_series(const double* q, double omega, int order, double* out) {
  su2_pow_series(q, omega, order, out);
}

void oracle_site_G_series(int nc, const double* K, double omega, int order, double* G) {
  store_mat(G, nc, site_G_series(load_mat(K, nc), omega, order, nc));
}

// One HALF sweep with the truncated-series power, in place (Landau gauge).
void oracle_or_sweep_series(const int32_t* dims, int nc, double* U, int parity, double omega, int order) {
  Lat L = make_lat(dims, nc);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) {
    if (parity_of(L, s) != parity) continue;
    Mat G = site_G_series(gather_K(U, L, s), omega, order, nc);
    Mat Gd = dagger(G, nc);
    for (int mu = 0; mu < 4; ++mu) {
      double* up = link_ptr(U, L, s, mu);
      store_mat(up, nc, mul(G, load_mat(up, nc), nc));
      double* dn = link_ptr(U, L, neighbour(L, s, mu, -1), mu);
      store_mat(dn, nc, mul(load_mat(dn, nc), Gd, nc));
    }
  }
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// Simulated annealing (named by the paper as the companion of overrelaxation, P:L7; its
// details are in the unavailable ref. [2] -- DESIGN.md reading C-25).
// Reading, from first principles: at temperature T the site's gauge transformation is not the
// maximiser of Re tr[g K(x)] but a sample of the Boltzmann weight exp(Re tr[g K(x)]/T) dg (Haar
// dg), per SU(2) subgroup for SU(3), with the same checkerboard, subgroup order and K <- g_s K,
// G <- g_s G bookkeeping as the overrelaxation sweep.  In a subgroup with quaternion p (as in
// subgroup_step) Re tr[g_s K] = |p| h_0 + const for h = q * (p/|p|), so h_0 has the density
// sqrt(1 - h_0^2) exp(a h_0), a = |p|/T, and the direction of the vector part of h is uniform on
// S^2; then q = h * conj(p)/|p|.  h_0 for a >= 2 by the Kennedy-Pendleton method:
//     lambda^2 = -( ln r1 + cos^2(2 pi r2) ln r3 ) / (2 a),  accept if r4^2 <= 1 - lambda^2,  h_0 = 1 - 2 lambda^2,
// and for a < 2 (where that method accepts too rarely) by Creutz's: h_0 = 1 + ln(x)/a with x uniform
// in [e^{-2a}, 1], accepted with probability sqrt(1 - h_0^2).
// Random numbers: the counter-based Philox4x32-10 generator (Salmon et al., SC'11), restated here;
// counter = (canonical site, half-sweep counter, subgroup | draw << 8, 0), key = 64-bit seed, so a
// site's numbers do not depend on the traversal order or the thread count.  Uniforms in (0,1):
// u = (w + 1/2) 2^-32 from each 32-bit word, one Philox block (4 uniforms) per trial / per direction.
// ---------------------------------------------------------------------------------------------
namespace {
void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
  uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
  uint32_t k0 = key_in[0], k1 = key_in[1];
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// four uniforms in (0,1) from one Philox block: u_i = (w_i + 1/2) 2^-32
void uniforms4(const uint32_t w[4], double u[4]) {
  for (int i = 0; i < 4; ++i) u[i] = ((double)w[i] + 0.5) * (1.0 / 4294967296.0);
}

struct SiteRng {
  uint32_t ctr[4];
  uint32_t key[2];
  uint32_t draw;
  void next4(double u[4]) {
    uint32_t c[4] = {ctr[0], ctr[1], ctr[2] | (draw << 8), ctr[3]};
    uint32_t w[4];
    philox4x32_10(c, key, w);
    uniforms4(w, u);
    ++draw;
  }
};

// q = h * conj(p)/|p| with h sampled as described above; a = |p|/T.
void su2_heatbath(const double p[4], double n, double T, SiteRng* rng, double q[4]) {
  const double a = n / T;
  double h0;
  if (a < 2.0) {
    // small a (hot / nearly cancelling K): Kennedy-Pendleton accepts with probability ~a^{3/2} there;
    // Creutz's method instead: x uniform in [e^{-2a}, 1], h_0 = 1 + ln(x)/a has density exp(a h_0)
    // on [-1, 1]; accept with probability sqrt(1 - h_0^2)
    const double emin = std::exp(-2.0 * a);
    for (;;) {
      double u[4];
      rng->next4(u);                                   // one block per trial (u[2], u[3] unused)
      double x = emin + u[0] * (1.0 - emin);
      h0 = 1.0 + std::log(x) / a;
      if (u[1] * u[1] <= 1.0 - h0 * h0) break;
    }
  } else {
    double lam2;
    for (;;) {
      double u[4];
      rng->next4(u);                                   // r1, r2, r3, r4: one block per trial
      double c = std::cos(2.0 * M_PI * u[1]);
      lam2 = -(std::log(u[0]) + c * c * std::log(u[2])) / (2.0 * a);
      if (u[3] * u[3] <= 1.0 - lam2) break;
    }
    h0 = 1.0 - 2.0 * lam2;
  }
  double u[4];
  rng->next4(u);                                     // direction of the vector part (u[2], u[3] unused)
  double ct = 2.0 * u[0] - 1.0;
  double st = std::sqrt(std::fmax(0.0, 1.0 - ct * ct));
  double phi = 2.0 * M_PI * u[1];
  double r = std::sqrt(std::fmax(0.0, 1.0 - h0 * h0));
  double h[4] = {h0, r * st * std::cos(phi), r * st * std::sin(phi), r * ct};
  // q = h * conj(p)/|p|   (quaternion product of convention C-7: (ab)_0 = a0 b0 - a.b, (ab)_v = a0 b + b0 a - a x b)
  double b[4] = {p[0] / n, -p[1] / n, -p[2] / n, -p[3] / n};
  q[0] = h[0] * b[0] - h[1] * b[1] - h[2] * b[2] - h[3] * b[3];
  q[1] = h[0] * b[1] + b[0] * h[1] - (h[2] * b[3] - h[3] * b[2]);
  q[2] = h[0] * b[2] + b[0] * h[2] - (h[3] * b[1] - h[1] * b[3]);
  q[3] = h[0] * b[3] + b[0] * h[3] - (h[1] * b[2] - h[2] * b[1]);
}

Mat site_G_heatbath(Mat K, double T, int nc, uint32_t site, uint32_t counter, uint64_t seed) {
  Mat G = unit_mat(nc);
  static const int pairs[3][2] = {{0, 1}, {0, 2}, {1, 2}};
  int npairs = (nc == 2) ? 1 : 3;
  for (int t = 0; t < npairs; ++t) {
    int i = pairs[t][0], j = pairs[t][1];
    double p[4] = {K.e[i][i].real() + K.e[j][j].real(), K.e[i][j].imag() + K.e[j][i].imag(),
                   K.e[i][j].real() - K.e[j][i].real(), K.e[i][i].imag() - K.e[j][j].imag()};
    double n = std::sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
    if (n == 0.0) continue;
    SiteRng rng;
    rng.ctr[0] = site; rng.ctr[1] = counter; rng.ctr[2] = (uint32_t)t; rng.ctr[3] = 0;
    rng.key[0] = (uint32_t)seed; rng.key[1] = (uint32_t)(seed >> 32);
    rng.draw = 0;
    double q[4];
    su2_heatbath(p, n, T, &rng, q);
    Mat gs = embed_su2(q, i, j, nc);
    K = mul(gs, K, nc);
    G = mul(gs, G, nc);
  }
  return G;
}

// ---- microcanonical step (SURVEY.md 8(f) NEXT-3 "simulated annealing + microcanonical steps";
// DESIGN.md reading C-26) ---------------------------------------------------------------------
// The energy-conserving companion of the heat bath: in each SU(2) subgroup the update is the
// REFLECTION q = g^2 of the maximiser g = conj(p)/|p| -- with h = q*p/|p| as in C-25 the local
// weight Re tr[g_s K] = |p| h_0 + const, and q = g^2 gives h = g, h_0 = p_0/|p|, the value q = 1
// gives as well: the functional is unchanged while the links move.  Written out as the quaternion
// square (c, v)^2 = (c^2 - v.v, 2 c v) (convention C-7; v x v = 0), no trigonometric function.
Mat site_G_micro(Mat K, int nc) {
  Mat G = unit_mat(nc);
  static const int pairs[3][2] = {{0, 1}, {0, 2}, {1, 2}};
  int npairs = (nc == 2) ? 1 : 3;
  for (int t = 0; t < npairs; ++t) {
    int i = pairs[t][0], j = pairs[t][1];
    double p[4] = {K.e[i][i].real() + K.e[j][j].real(), K.e[i][j].imag() + K.e[j][i].imag(),
                   K.e[i][j].real() - K.e[j][i].real(), K.e[i][i].imag() - K.e[j][j].imag()};
    double n = std::sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
    if (n == 0.0) continue;                                  // C-9
    double g[4] = {p[0] / n, -p[1] / n, -p[2] / n, -p[3] / n};
    double q[4] = {g[0] * g[0] - (g[1] * g[1] + g[2] * g[2] + g[3] * g[3]),
                   2.0 * g[0] * g[1], 2.0 * g[0] * g[2], 2.0 * g[0] * g[3]};
    Mat gs = embed_su2(q, i, j, nc);
    K = mul(gs, K, nc);
    G = mul(gs, G, nc);
  }
  return G;
}
}  // namespace

extern "C" {

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

// n samples of q for a given quaternion p at temperature T (site = sample index): out double[n][4].
void oracle_su2_heatbath_samples(const double* p, double T, uint64_t seed, int64_t n, double* out) {
  double nrm = std::sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  for (int64_t k = 0; k < n; ++k) {
    SiteRng rng;
    rng.ctr[0] = (uint32_t)k; rng.ctr[1] = 0; rng.ctr[2] = 0; rng.ctr[3] = 0;
    rng.key[0] = (uint32_t)seed; rng.key[1] = (uint32_t)(seed >> 32);
    rng.draw = 0;
    su2_heatbath(p, nrm, T, &rng, out + 4 * k);
  }
}

// One HALF sweep of simulated annealing at temperature T over the sites of `parity`, in place.
// `counter` must be different for every half-sweep of a run (it selects the random numbers).
void oracle_sa_sweep(const int32_t* dims, int nc, double* U, int parity, double T, uint64_t seed,
                     uint32_t counter) {
  Lat L = make_lat(dims, nc);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) {
    if (parity_of(L, s) != parity) continue;
    Mat G = site_G_heatbath(gather_K(U, L, s), T, nc, (uint32_t)s, counter, seed);
    Mat Gd = dagger(G, nc);
    for (int mu = 0; mu < 4; ++mu) {
      double* up = link_ptr(U, L, s, mu);
      store_mat(up, nc, mul(G, load_mat(up, nc), nc));
      double* dn = link_ptr(U, L, neighbour(L, s, mu, -1), mu);
      store_mat(dn, nc, mul(load_mat(dn, nc), Gd, nc));
    }
  }
}

// G of the microcanonical step for a given K (one site): K, G are double[nc][nc][2].
void oracle_site_G_micro(int nc, const double* K, double* G) {
  store_mat(G, nc, site_G_micro(load_mat(K, nc), nc));
}

// One microcanonical HALF sweep over the sites of `parity`, in place (reading C-26).
void oracle_micro_sweep(const int32_t* dims, int nc, double* U, int parity) {
  Lat L = make_lat(dims, nc);
#pragma omp parallel for num_threads(g_threads) schedule(static)
  for (int64_t s = 0; s < L.V; ++s) {
    if (parity_of(L, s) != parity) continue;
    Mat G = site_G_micro(gather_K(U, L, s), nc);
    Mat Gd = dagger(G, nc);
    for (int mu = 0; mu < 4; ++mu) {
      double* up = link_ptr(U, L, s, mu);
      store_mat(up, nc, mul(G, load_mat(up, nc), nc));
      double* dn = link_ptr(U, L, neighbour(L, s, mu, -1), mu);
      store_mat(dn, nc, mul(load_mat(dn, nc), Gd, nc));
    }
  }
}

}  // extern "C"
