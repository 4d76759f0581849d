// pslmc_host.h — host-side state shared by the translation units of libpslmc (not part of the ABI).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/pslmc.h"

namespace pslmc {

struct HostGroup {
  int stype = 0, ebin = 0;
  std::vector<uint16_t> ring, sector;
  std::vector<uint32_t> thresh, alias;
  double W = 0;
};

int fail(int code, const std::string &msg);
extern thread_local std::string g_error;

}  // namespace pslmc

// The opaque handle of the C ABI.
struct psl {
  int n_ebin = 0, n_ring = 0, n_sectors = 0;
  psr_params_t psr{};
  std::vector<double> W;
  jaws_t jaws{};
  std::vector<pslmc::HostGroup> groups;      // index = stype * n_ebin + ebin
  double rect[3][4] = {};
  // let shape: 0 = ring sectors (ring, sector), 1 = the paper's Cartesian grid (Xbin, Ybin) of square lets
  int let_mode = 0, n_xy = 0;
  double let_size = 0, grid_x0 = 0;
  // device tables (uploaded once)
  int device = -1;
  void *d_table = nullptr;                   // AliasEntry[total lets]
  uint32_t *d_let_off = nullptr, *d_n_let = nullptr;
  size_t total_lets = 0;
  // sigma_KN nodes in log2 E for photon energies up to the model's top energy (built once; layout: XsTable)
  void *d_xs = nullptr; double xs_x0 = 0, xs_h = 0;
  // Eq. 6 / Eq. 7 direction models (K = 0: focal geometry): DEVICE float4 {P_cum, mu, sigma_alpha, sigma_beta}[n_ebin][n_ring][K]
  void *d_dir[3] = {nullptr, nullptr, nullptr};
  int dir_K[3] = {0, 0, 0};
};

namespace pslmc {
int build_host(const psr_params_t &p, const jaws_t &j, int n_sectors, psl *out);
int build_host_grid(const psr_params_t &p, const jaws_t &j, double let_size, psl *out);
void allocate_host(const psl &P, uint64_t N, uint64_t *off);
int upload_tables(psl *P);                   // pslmc_dose.cu
}  // namespace pslmc
