// pslmc_psl.cu — host side of the source model: PSR→PSL conversion, sampling areas, alias tables,
// history allocation.  PAPER.md:35-57 §2.1.1 (Eq. 1-2), :61-69 §2.1.2, :75-80 S1-S2 (Eq. 3).
#include "pslmc_host.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <deque>

namespace pslmc {

thread_local std::string g_error;
int fail(int code, const std::string &msg) { g_error = msg; return code; }

static const double kPiD = 3.14159265358979323846;

// S1: sampling rectangle of a sub-source on the phase-space plane (Fig. 3 caption :69).
static void sampling_rect(const psr_params_t &p, const jaws_t &j, int stype, double r[4]) {
  if (stype == 0) {                       // primary photons: jaw opening scaled back to the plane
    const double s = p.z_phsp / j.sad;
    r[0] = j.x1 * s; r[1] = j.x2 * s; r[2] = j.y1 * s; r[3] = j.y2 * s;
    return;
  }
  // scattered photons and electrons: from the field centre on the iso plane back through the jaw
  // edges; the two jaw pairs sit at different z and are scaled separately, then intersected
  const double cx = 0.5 * (j.x1 + j.x2), cy = 0.5 * (j.y1 + j.y2);
  const double fx = (j.sad - p.z_phsp) / (j.sad - j.z_jx), fy = (j.sad - p.z_phsp) / (j.sad - j.z_jy);
  r[0] = cx + (j.x1 * j.z_jx / j.sad - cx) * fx;
  r[1] = cx + (j.x2 * j.z_jx / j.sad - cx) * fx;
  r[2] = cy + (j.y1 * j.z_jy / j.sad - cy) * fy;
  r[3] = cy + (j.y2 * j.z_jy / j.sad - cy) * fy;
}

// Does the bounding box of the annular sector touch the closed rectangle?  ("partially covered" lets)
static bool let_touches(double r0, double r1, double t0, double t1, const double rc[4]) {
  double xlo = 1e300, xhi = -1e300, ylo = 1e300, yhi = -1e300;
  auto add = [&](double x, double y) { xlo = std::min(xlo, x); xhi = std::max(xhi, x); ylo = std::min(ylo, y); yhi = std::max(yhi, y); };
  for (double r : {r0, r1}) for (double t : {t0, t1}) add(r * std::cos(t), r * std::sin(t));
  static const double ax[5] = {1, 0, -1, 0, 1}, ay[5] = {0, 1, 0, -1, 0};
  for (int k = 0; k <= 4; ++k) {
    const double ang = k * (kPiD / 2);
    if (ang >= t0 && ang <= t1) for (double r : {r0, r1}) add(r * ax[k], r * ay[k]);
  }
  return xlo <= rc[1] && xhi >= rc[0] && ylo <= rc[3] && yhi >= rc[2];
}

// Vose's alias method with FIFO work lists filled in ascending index (deterministic).
static void alias_table(const std::vector<double> &w, std::vector<uint32_t> &thresh, std::vector<uint32_t> &alias) {
  const size_t n = w.size();
  double sum = 0; for (double x : w) sum += x;
  std::vector<double> p(n), keep(n, 1.0);
  thresh.resize(n); alias.resize(n);
  std::deque<uint32_t> small, large;
  for (size_t i = 0; i < n; ++i) {
    p[i] = w[i] * (double)n / sum; alias[i] = (uint32_t)i;
    if (p[i] < 1.0) small.push_back((uint32_t)i); else large.push_back((uint32_t)i);
  }
  while (!small.empty() && !large.empty()) {
    const uint32_t s = small.front(), l = large.front();
    small.pop_front(); large.pop_front();
    keep[s] = p[s]; alias[s] = l;
    p[l] = (p[l] + p[s]) - 1.0;
    if (p[l] < 1.0) small.push_back(l); else large.push_back(l);
  }
  for (size_t i = 0; i < n; ++i) {
    if (keep[i] >= 1.0) { thresh[i] = 0xFFFFFFFFu; alias[i] = (uint32_t)i; continue; }
    const double t = std::floor(keep[i] * 4294967296.0);
    thresh[i] = (uint32_t)std::min(t, 4294967295.0);
  }
}

int build_host(const psr_params_t &p, const jaws_t &j, int n_sectors, psl *out) {
  out->n_ebin = p.n_ebin; out->n_ring = p.n_ring; out->n_sectors = n_sectors;
  out->psr = p; out->W.assign(p.W, p.W + (size_t)3 * p.n_ebin * p.n_ring); out->psr.W = nullptr;
  out->jaws = j;
  out->groups.assign((size_t)3 * p.n_ebin, HostGroup());
  bool any = false;
  for (int s = 0; s < 3; ++s) {
    sampling_rect(p, j, s, out->rect[s]);
    std::vector<uint16_t> ring, sector;
    for (int i = 0; i < p.n_ring; ++i)
      for (int k = 0; k < n_sectors; ++k)
        if (let_touches(i * p.ring_width, (i + 1) * p.ring_width, 2.0 * kPiD * k / n_sectors,
                        2.0 * kPiD * (k + 1) / n_sectors, out->rect[s])) { ring.push_back((uint16_t)i); sector.push_back((uint16_t)k); }
    for (int e = 0; e < p.n_ebin; ++e) {
      HostGroup &g = out->groups[(size_t)s * p.n_ebin + e];
      g.stype = s; g.ebin = e;
      std::vector<double> w;
      for (size_t a = 0; a < ring.size(); ++a) {
        const double wl = out->W[((size_t)s * p.n_ebin + e) * p.n_ring + ring[a]] / n_sectors;   // Eq. 1-2 over one sector
        if (wl > 0) { g.ring.push_back(ring[a]); g.sector.push_back(sector[a]); w.push_back(wl); }
      }
      g.W = 0; for (double x : w) g.W += x;
      if (!w.empty()) { alias_table(w, g.thresh, g.alias); any = true; }
    }
  }
  return any ? MC_OK : MC_E_EMPTY_FIELD;
}

// The paper's own let shape: a Cartesian grid of square lets of side `a` over the phase-space
// disc.  Weight of let (Xbin, Ybin), steps 1-4: radius of the let centre; ring weight at that radius by linear
// interpolation between ring centres (towards (0, 0) inside the first centre, constant beyond the last); divided by
// 2 pi r; one normalisation over all lets of all energies and sub-sources.  A let is active when any portion of
// its square lies in the closed sampling rectangle (:69).  HostGroup::ring / ::sector hold Xbin / Ybin.
static double grid_weight(const double *W, int n_ring, double dr, double r) {
  const double t = r / dr - 0.5;
  double w;
  if (t <= 0) w = W[0] * (r / (0.5 * dr));             // towards (0, 0): a ring of radius 0 holds nothing
  else if (t >= n_ring - 1) w = W[n_ring - 1];
  else { const int i = (int)std::floor(t); const double f = t - i; w = W[i] + f * (W[i + 1] - W[i]); }
  return w / (2.0 * kPiD * r);
}

int build_host_grid(const psr_params_t &p, const jaws_t &j, double a, psl *out) {
  out->n_ebin = p.n_ebin; out->n_ring = p.n_ring; out->n_sectors = 0;
  out->psr = p; out->W.assign(p.W, p.W + (size_t)3 * p.n_ebin * p.n_ring); out->psr.W = nullptr;
  out->jaws = j;
  out->groups.assign((size_t)3 * p.n_ebin, HostGroup());
  const double rmax = p.n_ring * p.ring_width;
  const int half = (int)std::ceil(rmax / a);             // even number of lets per side: no centre on the axis
  out->let_mode = 1; out->let_size = a; out->n_xy = 2 * half; out->grid_x0 = -half * a;
  const int n = out->n_xy;
  // radius of every let centre, once
  std::vector<double> rad((size_t)n * n);
  for (int X = 0; X < n; ++X) for (int Y = 0; Y < n; ++Y) {
    const double x = out->grid_x0 + (X + 0.5) * a, y = out->grid_x0 + (Y + 0.5) * a;
    rad[(size_t)X * n + Y] = std::sqrt(x * x + y * y);
  }
  double total = 0;
  for (int s = 0; s < 3; ++s) for (int e = 0; e < p.n_ebin; ++e) {
    const double *Wr = &out->W[((size_t)s * p.n_ebin + e) * p.n_ring];
    for (int X = 0; X < n; ++X) for (int Y = 0; Y < n; ++Y) {
      const double r = rad[(size_t)X * n + Y];
      if (r < rmax) total += grid_weight(Wr, p.n_ring, p.ring_width, r);
    }
  }
  bool any = false;
  for (int s = 0; s < 3; ++s) {
    sampling_rect(p, j, s, out->rect[s]);
    const double *rc = out->rect[s];
    for (int e = 0; e < p.n_ebin; ++e) {
      HostGroup &g = out->groups[(size_t)s * p.n_ebin + e];
      g.stype = s; g.ebin = e;
      const double *Wr = &out->W[((size_t)s * p.n_ebin + e) * p.n_ring];
      std::vector<double> w;
      for (int X = 0; X < n; ++X) for (int Y = 0; Y < n; ++Y) {
        const double r = rad[(size_t)X * n + Y];
        if (!(r < rmax)) continue;
        const double xl = out->grid_x0 + X * a, yl = out->grid_x0 + Y * a;
        if (!(xl <= rc[1] && xl + a >= rc[0] && yl <= rc[3] && yl + a >= rc[2])) continue;
        const double wl = grid_weight(Wr, p.n_ring, p.ring_width, r) / total;
        if (wl > 0) { g.ring.push_back((uint16_t)X); g.sector.push_back((uint16_t)Y); w.push_back(wl); }
      }
      g.W = 0; for (double x : w) g.W += x;
      if (!w.empty()) { alias_table(w, g.thresh, g.alias); any = true; }
    }
  }
  return any ? MC_OK : MC_E_EMPTY_FIELD;
}

// Eq. 3 at group level, largest-remainder rounding, ties to the lower group index.
void allocate_host(const psl &P, uint64_t N, uint64_t *off) {
  const size_t G = P.groups.size();
  double tot = 0; for (const HostGroup &g : P.groups) tot += g.W;
  std::vector<uint64_t> n(G); std::vector<double> frac(G);
  uint64_t used = 0;
  for (size_t g = 0; g < G; ++g) {
    const double q = (double)N * P.groups[g].W / tot, f = std::floor(q);
    n[g] = (uint64_t)f; frac[g] = q - f; used += n[g];
  }
  std::vector<size_t> order(G);
  for (size_t g = 0; g < G; ++g) order[g] = g;
  std::stable_sort(order.begin(), order.end(), [&](size_t a, size_t b) { return frac[a] > frac[b]; });
  const uint64_t rem = used <= N ? N - used : 0;      // N <= 2^53 (checked by the callers): (double)N is exact and used <= N
  for (uint64_t r = 0; r < rem; ++r) ++n[order[r % G]];
  off[0] = 0;
  for (size_t g = 0; g < G; ++g) off[g + 1] = off[g] + n[g];
}

}  // namespace pslmc

using namespace pslmc;

extern "C" int psl_build(const psr_params_t *psr, const jaws_t *jaws, int32_t n_sectors, psl_t **out) {
  if (!psr || !jaws || !out || !psr->W || psr->n_ebin < 1 || psr->n_ring < 1 || n_sectors < 1 || n_sectors > 65535 ||
      psr->n_ring > 65535 || 3 * psr->n_ebin > 159 || !(jaws->x1 < jaws->x2) || !(jaws->y1 < jaws->y2) ||
      !(psr->ring_width > 0) || !(psr->e_bin_width > 0))
    return fail(MC_E_INVALID_ARG, "psl_build: invalid argument");
  if (!(psr->e_min >= 0) || !(psr->e_min + psr->n_ebin * psr->e_bin_width < 4096.0))     // the exact warp sums of the ledgers hold energies below 4096 MeV
    return fail(MC_E_INVALID_ARG, "psl_build: energy range must lie in [0, 4096) MeV");
  for (int s = 0; s < 3; ++s)
    if (!(psr->z_phsp > psr->z_src[s]) || !(jaws->z_jx > psr->z_src[s]) || !(jaws->z_jy > psr->z_src[s]) || psr->sigma_src[s] < 0 ||
        (psr->particle_type[s] != 0 && psr->particle_type[s] != 1))
      return fail(MC_E_INVALID_ARG, "psl_build: sub-source geometry invalid");
  psl *P = new psl();
  int rc = build_host(*psr, *jaws, n_sectors, P);
  if (rc != MC_OK) { delete P; return fail(rc, "psl_build: no let is active for this jaw setting"); }
  rc = upload_tables(P);
  if (rc != MC_OK) { psl_free(P); return rc; }
  *out = P;
  return MC_OK;
}

extern "C" int psl_build_grid(const psr_params_t *psr, const jaws_t *jaws, double let_size, psl_t **out) {
  if (!psr || !jaws || !out || !psr->W || psr->n_ebin < 1 || psr->n_ring < 1 || psr->n_ring > 65535 || 3 * psr->n_ebin > 159 ||
      !(jaws->x1 < jaws->x2) || !(jaws->y1 < jaws->y2) || !(psr->ring_width > 0) || !(psr->e_bin_width > 0) || !(let_size > 0) ||
      2.0 * std::ceil(psr->n_ring * psr->ring_width / let_size) > 4096.0)
    return fail(MC_E_INVALID_ARG, "psl_build_grid: invalid argument");
  if (!(psr->e_min >= 0) || !(psr->e_min + psr->n_ebin * psr->e_bin_width < 4096.0))
    return fail(MC_E_INVALID_ARG, "psl_build_grid: energy range must lie in [0, 4096) MeV");
  for (int s = 0; s < 3; ++s)
    if (!(psr->z_phsp > psr->z_src[s]) || !(jaws->z_jx > psr->z_src[s]) || !(jaws->z_jy > psr->z_src[s]) || psr->sigma_src[s] < 0 ||
        (psr->particle_type[s] != 0 && psr->particle_type[s] != 1))
      return fail(MC_E_INVALID_ARG, "psl_build_grid: sub-source geometry invalid");
  psl *P = new psl();
  int rc = build_host_grid(*psr, *jaws, let_size, P);
  if (rc != MC_OK) { delete P; return fail(rc, "psl_build_grid: no let is active for this jaw setting"); }
  rc = upload_tables(P);
  if (rc != MC_OK) { psl_free(P); return rc; }
  *out = P;
  return MC_OK;
}

extern "C" int psl_allocate(const psl_t *P, uint64_t n_histories, uint64_t *off_out) {
  if (!P || !off_out) return fail(MC_E_INVALID_ARG, "psl_allocate: null argument");
  if (n_histories > (1ull << 53)) return fail(MC_E_INVALID_ARG, "psl_allocate: n_histories above 2^53 (Eq. 3 is evaluated in double)");
  allocate_host(*P, n_histories, off_out);
  return MC_OK;
}

// Eq. 3 across the beams of a plan (the denominator runs over the sampling areas of ALL beams):
// beam i gets N * W_i / sum_j W_j histories, W_i = sum of its active group weights, largest-remainder rounding,
// ties to the lower beam index.
extern "C" int mc_plan_allocate(const psl_t *const *psls, int32_t n_beams, uint64_t n_histories, uint64_t *n_out) {
  if (!psls || !n_out || n_beams < 1 || n_histories > (1ull << 53)) return fail(MC_E_INVALID_ARG, "mc_plan_allocate: invalid argument (n_histories <= 2^53)");
  std::vector<double> W(n_beams, 0.0), frac(n_beams);
  double tot = 0;
  for (int i = 0; i < n_beams; ++i) {
    if (!psls[i]) return fail(MC_E_INVALID_ARG, "mc_plan_allocate: null beam");
    for (const HostGroup &g : psls[i]->groups) W[i] += g.W;
    tot += W[i];
  }
  if (!(tot > 0)) return fail(MC_E_EMPTY_FIELD, "mc_plan_allocate: no active let in any beam");
  uint64_t used = 0;
  for (int i = 0; i < n_beams; ++i) {
    const double q = (double)n_histories * W[i] / tot, f = std::floor(q);
    n_out[i] = (uint64_t)f; frac[i] = q - f; used += n_out[i];
  }
  std::vector<int> order(n_beams);
  for (int i = 0; i < n_beams; ++i) order[i] = i;
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return frac[a] > frac[b]; });
  const uint64_t rem = used <= n_histories ? n_histories - used : 0;
  for (uint64_t r = 0; r < rem; ++r) ++n_out[order[r % n_beams]];
  return MC_OK;
}

extern "C" int psl_export(const psl_t *P, void *host_buf, size_t *bytes) {
  if (!P || !bytes) return fail(MC_E_INVALID_ARG, "psl_export: null argument");
  auto pad8 = [](size_t b) { return (b + 7) & ~(size_t)7; };
  size_t need = 8;
  for (const HostGroup &g : P->groups) need += 24 + 2 * pad8(2 * g.ring.size()) + 2 * pad8(4 * g.ring.size());
  need += sizeof(double) * 12;
  if (!host_buf) { *bytes = need; return MC_OK; }
  if (*bytes < need) return fail(MC_E_INVALID_ARG, "psl_export: buffer too small");
  char *o = (char *)host_buf;
  std::memset(o, 0, need);
  auto put = [&](const void *src, size_t b) { std::memcpy(o, src, b); o += pad8(b); };
  const uint64_t G = P->groups.size(); put(&G, 8);
  for (const HostGroup &g : P->groups) {
    const int32_t hdr[2] = {g.stype, g.ebin}; const uint64_t n = g.ring.size();
    put(hdr, 8); put(&n, 8); put(&g.W, 8);
    put(g.ring.data(), 2 * n); put(g.sector.data(), 2 * n); put(g.thresh.data(), 4 * n); put(g.alias.data(), 4 * n);
  }
  put(P->rect, sizeof(double) * 12);
  *bytes = need;
  return MC_OK;
}

extern "C" const char *mc_last_error(void) { return g_error.c_str(); }
