// Harness for tests/test_oracle_sanitized.py: includes the oracle's translation unit and drives
// every exported function once on a small asymmetric lattice, so that the whole file can be run
// under -fsanitize=address,undefined.  Inputs are arbitrary finite matrices:
// memory safety does not depend on unitarity.
#include "../oracle/oracle.cpp"

#include <cstdio>

int main() {
  const int32_t dims[4] = {4, 6, 2, 8};
  const int64_t V = 4 * 6 * 2 * 8;
  uint64_t state = 88172645463325252ull;
  auto rnd = [&]() {
    state ^= state << 13; state ^= state >> 7; state ^= state << 17;
    return (double)(state >> 11) / 9007199254740992.0 - 0.5;
  };
  for (int nc = 2; nc <= 3; ++nc) {
    const size_t n = (size_t)V * 4 * nc * nc * 2;
    std::vector<double> U(n), K((size_t)V * nc * nc * 2), D(K.size()), g(K.size());
    for (auto& x : U) x = rnd();
    for (auto& x : g) x = rnd();
    oracle_reunitarize(V * 4, nc, U.data());
    oracle_reunitarize(V, nc, g.data());
    oracle_set_threads(2);
    oracle_K(dims, nc, U.data(), K.data());
    oracle_delta(dims, nc, U.data(), D.data());
    oracle_K_coulomb(dims, nc, U.data(), K.data());
    oracle_delta_coulomb(dims, nc, U.data(), D.data());
    std::vector<double> G(nc * nc * 2), gs(nc * nc * 2);
    oracle_site_G(nc, K.data(), 1.7, G.data());
    oracle_site_G_series(nc, K.data(), 1.7, 4, G.data());
    oracle_subgroup_step(nc, K.data(), 0, 1, 1.7, gs.data());
    for (int parity = 0; parity < 2; ++parity) {
      oracle_or_sweep(dims, nc, U.data(), parity, 1.7);
      oracle_or_sweep_coulomb(dims, nc, U.data(), parity, 1.7);
      oracle_or_sweep_series(dims, nc, U.data(), parity, 1.7, 5);
      oracle_sa_sweep(dims, nc, U.data(), parity, 0.5, 42ull, (uint32_t)parity);
    }
    oracle_gauge_transform(dims, nc, U.data(), g.data());
    std::vector<double> th(dims[3]), F(dims[3]);
    oracle_coulomb_theta_F(dims, nc, U.data(), th.data(), F.data());
    double a = oracle_functional(dims, nc, U.data()) + oracle_gauge_precision(dims, nc, U.data()) +
               oracle_plaquette(dims, nc, U.data()) + th[0] + F[dims[3] - 1];
    if (nc == 3) oracle_reconstruct12(V * 4, U.data());
    double q[4] = {0.6, 0.0, 0.8, 0.0}, out[4];
    oracle_su2_pow(q, 1.7, out);
    oracle_su2_pow_series(q, 1.7, 6, out);
    std::vector<double> samples(4 * 100);
    oracle_su2_heatbath_samples(q, 0.3, 7ull, 100, samples.data());
    uint32_t ctr[4] = {1, 2, 3, 4}, key[2] = {5, 6}, w[4];
    oracle_philox4x32_10(ctr, key, w);
    std::printf("nc=%d ok %.6f %u %d\n", nc, a + out[0] + samples[0], w[0], oracle_max_threads());
  }
  return 0;
}
