// pslmc_oracle.cpp — the ORACLE: a plain, slow, single-threaded, double-precision CPU statement of
// what the PSL source + Monte Carlo dose hot path computes.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference leg may build, load or call it.  It shares no code,
// header, table or constant generator with paper_1503_01725_b200/csrc (the CUDA path); the
// constants below are typed here independently.
//
// What it follows (PAPER.md = arxiv 1503.01725; DESIGN.md §"Readings" fixes what the paper leaves
// open — the paper gives no transport physics, BASELINE.json's north_star prescribes the analytic set):
//   philox_block        DESIGN.md R1  (Philox4x32-10, Salmon et al. SC'11; keyed by seed, history)
//   psl_build           PAPER.md:41-55 Eq. 1-2 (ring → let weights), :61-69 §2.1.2 (sampling areas)
//   psl_build_grid      PAPER.md:39-55 steps 1-4: the paper's own Cartesian (Xbin, Ybin) let grid (NEXT-1)
//   allocate            PAPER.md:76-80 Eq. 3 (group level, largest remainder)
//   sample_history      PAPER.md:82-92 S3 Eq. 4-5, :94-116 S4-S5 (focal geometry reading, or Eq. 6-7 as printed: NEXT-2), jaws :65/:92
//   photon / electron   PAPER.md:161 (cut-offs); P1-P9 (Woodcock, Kahn, CSDA + Gaussian MS)
//   deposit / ledgers   DESIGN.md S1 (int64 fixed point, 2^-32 MeV); commissioning tally PAPER.md:132-138 (NEXT-3)
//   fingerprints        DESIGN.md F1 (plain: the interaction sequence; FLAG_FP_VOXELS: the strict form used by the every-voxel parity test)
//   orc_dose_list       the same path over a LIST of history ids (the tally of the diverged histories in that test); no arithmetic of its own
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Philox vs cuRAND's host generator; ring/sector
// weights vs closed forms; alias reconstruction; chi-square of sampled spectrum / fluence vs the
// analytic PSR densities; source back-projection Gaussian; Klein–Nishina angular chi-square and
// total cross-section vs quadrature of the differential; interaction fractions; exp(-mu x)
// transmission (homogeneous and layered); CSDA path length vs the closed-form integral; Highland
// angle moments; energy conservation; permutation invariance; single-history hand trace; Compton recoil electron by
// momentum conservation, pair energy split and annihilation-photon geometry (tests/test_oracle_secondaries.py).
// No function here is "parity unpinned" (child_track and orc_com_column are [proposed] numberings with nothing
// external to check against: they are pinned for determinism and by-hand values only).
//
// Build: g++ -O2 -std=c++17 -shared -fPIC (no -ffast-math, no -march) — see oracle/__init__.py.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <deque>
#include <limits>
#include <vector>

namespace {

typedef unsigned __int128 u128;
typedef __int128 i128;

// ---------------------------------------------------------------- constants (DESIGN.md tables)
const double PI = 3.14159265358979323846;
const double ME = 0.51099895;          // electron rest energy, MeV (Compton alpha, p*beta)
const double RE2 = 7.940787e-26;       // classical electron radius squared, cm^2
const double E_PAIR = 1.022;           // pair threshold and annihilation total, MeV
const double E_ANNIH = 0.511;          // each annihilation photon, MeV
const double PCUT = 0.05;              // photon cut-off, MeV
const double ECUT = 0.2;               // electron cut-off, MeV
const double EPS_B = 1e-4;             // boundary nudge, cm
const double NE[3] = {3.343e23, 3.343e23, 3.100e23};      // electrons per gram: water, lung, bone
const double CPHOTO[3] = {2.77e-6, 2.77e-6, 2.2e-5};      // photo-electric, cm^2 g^-1 MeV^3
const double PPAIR[3] = {9.6e-4, 9.6e-4, 1.3e-3};         // pair, cm^2 g^-1
const double SSCALE[3] = {1.0, 1.0, 0.92};                // stopping-power scale
const double X0[3] = {36.08, 36.08, 27.2};                // radiation length, g cm^-2
const double FE_DEFAULT = 0.12;                           // energy-loss fraction per step
const double FIX = 4294967296.0;                          // 2^32 quanta per MeV

const int FLAG_ELECTRONS_LOCAL = 1;
const int FLAG_TRACE_BIRTH = 2;       // orc_trace only: log a 'B' event (position, direction, energy) when a track starts
const int FLAG_FP_VOXELS = 4;         // strict fingerprints (F1): also the voxel of every deposit, the stream position after every
                                      // accepted Kahn sampling (= which trial was accepted) with the branch it took, and whether an electron sub-step ended its condensed step

// ---------------------------------------------------------------- R1: Philox4x32-10
void philox_block(uint64_t seed, uint64_t h, uint32_t track, uint32_t block, uint32_t out[4]) {
  uint32_t c0 = block, c1 = track, c2 = (uint32_t)h, c3 = (uint32_t)(h >> 32);
  uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// The stream of a track (seed, history, track) is its sequence of Philox blocks 0, 1, 2, ...  Every EVENT of the
// track takes the next whole block and uses its first words in the order stated at the event; the words it does
// not use are discarded (R1).  `j` = the next block.
struct Stream {
  uint64_t seed, h; uint32_t track, j;
  void next_block(uint32_t w[4]) { philox_block(seed, h, track, j++, w); }
};
inline double U_co(uint32_t x) { return (double)(x >> 8) * (1.0 / 16777216.0); }          // [0,1)
inline double U_oc(uint32_t x) { return (double)((x >> 8) + 1) * (1.0 / 16777216.0); }    // (0,1]

inline uint32_t child_track(uint32_t parent, uint32_t n, uint32_t c) {
  return (((parent ^ 0x9E3779B9u) * 0x01000193u) ^ ((n << 2) | c)) * 0x01000193u;
}

// ---------------------------------------------------------------- F1: FNV-1a-64 fingerprints
struct Fnv {
  uint64_t v = 0xcbf29ce484222325ull;
  void byte(uint8_t b) { v = (v ^ b) * 0x100000001b3ull; }
  void u32(uint32_t x) { for (int i = 0; i < 4; ++i) byte((uint8_t)(x >> (8 * i))); }
};

// ---------------------------------------------------------------- plain structs of the C API
struct PsrParams {
  int32_t n_ebin, n_ring; double e_min, e_bin_width, ring_width, z_phsp; const double *W;
  double sigma_src[3], z_src[3]; int32_t particle_type[3];
};
struct Jaws { double x1, x2, y1, y2, z_jx, z_jy, sad; };
struct Phantom { int32_t nx, ny, nz; double dx, dy, dz, ox, oy, oz; const float *density; const uint8_t *material; };
struct Beam { double iso[3]; double R[9]; double sad; };
struct Result {
  int64_t ledger_hi[4]; uint64_t ledger_lo[4];   // incident, deposited, escaped, jaw
  uint64_t n_hist[3]; uint64_t n_jaw_rejected;
  uint64_t n_missed, n_flights, n_virtual, n_compton, n_photo, n_pair;
  uint64_t n_photon_cutoff, n_photon_escape, n_uncollided_escape;
  uint64_t n_sec_electrons, n_sec_photons;
  uint64_t n_electron_tracks, n_electron_steps, n_electron_escape;
  uint64_t n_deposits;
  uint64_t n_kahn_trials, n_deflections;   // work counters (bench.py's algorithmic-work numerator): Kahn trials, condensed-step deflections
};

struct Group { int stype, ebin; std::vector<uint16_t> ring, sector; std::vector<uint32_t> thresh, alias; double W = 0; };
struct Psl {
  PsrParams p; std::vector<double> Wcopy; Jaws jaws; int n_sectors;
  std::vector<Group> groups;     // index = stype * n_ebin + ebin
  double rect[3][4];             // xlo, xhi, ylo, yhi per sub-source
  // Cartesian (Xbin, Ybin) let grid of PAPER.md:39-55 (mode 1): n_xy x n_xy square lets of side let_size,
  // lower-left corner of let (0,0) at (grid_x0, grid_x0); Group::ring holds Xbin, Group::sector holds Ybin.
  int mode = 0, n_xy = 0; double let_size = 0, grid_x0 = 0;
  // Direction models of PAPER.md:94-116 (Eq. 6: K Gaussians in (alpha, beta) per (energy bin, ring); Eq. 7: K = 1,
  // mean 0), one per sub-source, K = 0 = the focal-geometry model.  Arrays [n_ebin][n_ring][K]; P = the cumulative
  // look-up table P_{i,k} = sum_{j<=k} c_{i,j} / sum_{j<=K} c_{i,j}  (:107 with the denominator read as the full sum).
  struct DirModel { int K = 0; std::vector<double> P, mu, sa, sb; } dir[3];
};

// ---------------------------------------------------------------- psl_build
// Sampling rectangle on the phase-space plane (Fig. 3 caption :69).
void sampling_rect(const PsrParams &p, const Jaws &j, int stype, double r[4]) {
  if (stype == 0) {  // primary: jaw opening scaled back to the phase-space plane
    double s = p.z_phsp / j.sad;
    r[0] = j.x1 * s; r[1] = j.x2 * s; r[2] = j.y1 * s; r[3] = j.y2 * s;
  } else {           // scattered photons, electrons: back-project from the field centre through
                     // the jaw edges (upper surface), x and y pairs at their own z
    double cx = 0.5 * (j.x1 + j.x2), cy = 0.5 * (j.y1 + j.y2);
    double fx = (j.sad - p.z_phsp) / (j.sad - j.z_jx), fy = (j.sad - p.z_phsp) / (j.sad - j.z_jy);
    r[0] = cx + (j.x1 * j.z_jx / j.sad - cx) * fx;
    r[1] = cx + (j.x2 * j.z_jx / j.sad - cx) * fx;
    r[2] = cy + (j.y1 * j.z_jy / j.sad - cy) * fy;
    r[3] = cy + (j.y2 * j.z_jy / j.sad - cy) * fy;
  }
}

// Axis-aligned bounding box of the annular sector r in [r0,r1], theta in [t0,t1].
void sector_bbox(double r0, double r1, double t0, double t1, double bb[4]) {
  double xs[12], ys[12]; int n = 0;
  const double rr[2] = {r0, r1}, tt[2] = {t0, t1};
  for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) { xs[n] = rr[a] * std::cos(tt[b]); ys[n] = rr[a] * std::sin(tt[b]); ++n; }
  for (int k = 0; k <= 4; ++k) {          // axis directions k*pi/2 that fall inside the sector
    double ang = k * (PI / 2);
    if (ang >= t0 && ang <= t1) {
      const double cx[5] = {1, 0, -1, 0, 1}, cy[5] = {0, 1, 0, -1, 0};
      for (int a = 0; a < 2; ++a) { xs[n] = rr[a] * cx[k]; ys[n] = rr[a] * cy[k]; ++n; }
    }
  }
  bb[0] = bb[1] = xs[0]; bb[2] = bb[3] = ys[0];
  for (int i = 1; i < n; ++i) {
    if (xs[i] < bb[0]) bb[0] = xs[i]; if (xs[i] > bb[1]) bb[1] = xs[i];
    if (ys[i] < bb[2]) bb[2] = ys[i]; if (ys[i] > bb[3]) bb[3] = ys[i];
  }
}

// Vose's alias method made deterministic (A1).
void build_alias(const std::vector<double> &w, std::vector<uint32_t> &thresh, std::vector<uint32_t> &alias) {
  size_t n = w.size();
  thresh.assign(n, 0); alias.assign(n, 0);
  double sum = 0; for (size_t i = 0; i < n; ++i) sum += w[i];
  std::vector<double> p(n), pt(n, 1.0);
  std::deque<uint32_t> small, large;
  for (size_t i = 0; i < n; ++i) { p[i] = w[i] * (double)n / sum; alias[i] = (uint32_t)i; (p[i] < 1.0 ? small : large).push_back((uint32_t)i); }
  while (!small.empty() && !large.empty()) {
    uint32_t s = small.front(); small.pop_front();
    uint32_t l = large.front(); large.pop_front();
    pt[s] = p[s]; alias[s] = l;
    p[l] = (p[l] + p[s]) - 1.0;
    (p[l] < 1.0 ? small : large).push_back(l);
  }
  // leftovers keep pt = 1, alias = self
  for (size_t i = 0; i < n; ++i) {
    double t = std::floor(pt[i] * FIX);
    if (pt[i] >= 1.0) { thresh[i] = 0xFFFFFFFFu; alias[i] = (uint32_t)i; }
    else thresh[i] = (uint32_t)(t > 4294967295.0 ? 4294967295.0 : t);
  }
}

Psl *psl_build(const PsrParams &p, const Jaws &j, int n_sectors) {
  Psl *psl = new Psl;
  psl->p = p; psl->jaws = j; psl->n_sectors = n_sectors;
  psl->Wcopy.assign(p.W, p.W + (size_t)3 * p.n_ebin * p.n_ring);
  psl->p.W = psl->Wcopy.data();
  psl->groups.resize((size_t)3 * p.n_ebin);
  bool any = false;
  for (int s = 0; s < 3; ++s) {
    sampling_rect(p, j, s, psl->rect[s]);
    const double *rc = psl->rect[s];
    // active lets of this sub-source, (ring, sector) order
    std::vector<uint16_t> ring, sector;
    for (int i = 0; i < p.n_ring; ++i)
      for (int k = 0; k < n_sectors; ++k) {
        double bb[4];
        sector_bbox(i * p.ring_width, (i + 1) * p.ring_width, 2.0 * PI * k / n_sectors, 2.0 * PI * (k + 1) / n_sectors, bb);
        bool overlap = bb[0] <= rc[1] && bb[1] >= rc[0] && bb[2] <= rc[3] && bb[3] >= rc[2];
        if (overlap) { ring.push_back((uint16_t)i); sector.push_back((uint16_t)k); }
      }
    for (int e = 0; e < p.n_ebin; ++e) {
      Group &g = psl->groups[(size_t)s * p.n_ebin + e];
      g.stype = s; g.ebin = e;
      std::vector<double> w;
      for (size_t a = 0; a < ring.size(); ++a) {
        double wl = psl->Wcopy[((size_t)s * p.n_ebin + e) * p.n_ring + ring[a]] / n_sectors;   // Eq. 1-2 over a sector
        if (wl > 0) { g.ring.push_back(ring[a]); g.sector.push_back(sector[a]); w.push_back(wl); }
      }
      g.W = 0; for (double x : w) g.W += x;
      if (!w.empty()) { build_alias(w, g.thresh, g.alias); any = true; }
    }
  }
  if (!any) { delete psl; return nullptr; }
  return psl;
}

// PAPER.md:55 steps 1-4: weight of the square let centred at radius r from the ring weights W[0..n_ring):
// step 2 = linear interpolation of W_Rbin along the radius between ring centres (i + 1/2) dr; inside the first
// centre between (0, 0) and (dr/2, W_0) - a ring of radius 0 holds no particles, and any other anchor makes
// W/(2 pi r) diverge on the axis - and held constant beyond the last centre (A3 reading);
// step 3 = divide by 2 pi r.
double grid_let_weight(const double *W, int n_ring, double dr, double r) {
  double t = r / dr - 0.5;                        // position in units of ring centres
  double w;
  if (t <= 0) w = W[0] * (r / (0.5 * dr));
  else if (t >= n_ring - 1) w = W[n_ring - 1];
  else { int i = (int)std::floor(t); double f = t - i; w = W[i] + f * (W[i + 1] - W[i]); }
  return w / (2.0 * PI * r);
}

// PSR -> PSL on the paper's Cartesian grid (Eq. 1-2, steps 1-4) + sampling areas (:61-69).
Psl *psl_build_grid(const PsrParams &p, const Jaws &j, double let_size) {
  Psl *psl = new Psl;
  psl->p = p; psl->jaws = j; psl->n_sectors = 0; psl->mode = 1; psl->let_size = let_size;
  psl->Wcopy.assign(p.W, p.W + (size_t)3 * p.n_ebin * p.n_ring);
  psl->p.W = psl->Wcopy.data();
  psl->groups.resize((size_t)3 * p.n_ebin);
  const double rmax = p.n_ring * p.ring_width;
  const int half = (int)std::ceil(rmax / let_size);      // an even number of lets per side: no let centre on the axis
  psl->n_xy = 2 * half; psl->grid_x0 = -half * let_size;
  // step 4: one normalisation over all lets of all energies and sub-sources
  double total = 0;
  for (int s = 0; s < 3; ++s) for (int e = 0; e < p.n_ebin; ++e)
    for (int X = 0; X < psl->n_xy; ++X) for (int Y = 0; Y < psl->n_xy; ++Y) {
      double x = psl->grid_x0 + (X + 0.5) * let_size, y = psl->grid_x0 + (Y + 0.5) * let_size, r = std::sqrt(x * x + y * y);   // step 1
      if (r < rmax) total += grid_let_weight(&psl->Wcopy[((size_t)s * p.n_ebin + e) * p.n_ring], p.n_ring, p.ring_width, r);
    }
  bool any = false;
  for (int s = 0; s < 3; ++s) {
    sampling_rect(p, j, s, psl->rect[s]);
    const double *rc = psl->rect[s];
    for (int e = 0; e < p.n_ebin; ++e) {
      Group &g = psl->groups[(size_t)s * p.n_ebin + e];
      g.stype = s; g.ebin = e;
      std::vector<double> w;
      for (int X = 0; X < psl->n_xy; ++X) for (int Y = 0; Y < psl->n_xy; ++Y) {
        double xl = psl->grid_x0 + X * let_size, yl = psl->grid_x0 + Y * let_size;
        double x = xl + 0.5 * let_size, y = yl + 0.5 * let_size, r = std::sqrt(x * x + y * y);
        if (!(r < rmax)) continue;                               // outside the model's phase-space disc
        bool overlap = xl <= rc[1] && xl + let_size >= rc[0] && yl <= rc[3] && yl + let_size >= rc[2];   // "any portion" (:69)
        if (!overlap) continue;
        double wl = grid_let_weight(&psl->Wcopy[((size_t)s * p.n_ebin + e) * p.n_ring], p.n_ring, p.ring_width, r) / total;
        if (wl > 0) { g.ring.push_back((uint16_t)X); g.sector.push_back((uint16_t)Y); w.push_back(wl); }
      }
      g.W = 0; for (double x : w) g.W += x;
      if (!w.empty()) { build_alias(w, g.thresh, g.alias); any = true; }
    }
  }
  if (!any) { delete psl; return nullptr; }
  return psl;
}

// Eq. 3 at group level with largest-remainder rounding (A2).
void allocate(const Psl &psl, uint64_t N, uint64_t *off) {
  size_t G = psl.groups.size();
  double tot = 0; for (size_t g = 0; g < G; ++g) tot += psl.groups[g].W;
  std::vector<uint64_t> n(G); std::vector<double> frac(G);
  uint64_t used = 0;
  for (size_t g = 0; g < G; ++g) {
    double q = (double)N * psl.groups[g].W / tot;
    double f = std::floor(q);
    n[g] = (uint64_t)f; frac[g] = q - f; used += n[g];
  }
  // hand the N - used leftover histories to the largest fractional parts, ties to the lower index
  std::vector<size_t> idx(G);
  for (size_t g = 0; g < G; ++g) idx[g] = g;
  std::stable_sort(idx.begin(), idx.end(), [&](size_t a, size_t b) { return frac[a] > frac[b]; });
  uint64_t rem = N - used;                       // < G: every fractional part is < 1
  for (uint64_t r = 0; r < rem; ++r) ++n[idx[r % G]];
  off[0] = 0; for (size_t g = 0; g < G; ++g) off[g + 1] = off[g] + n[g];
}

// ---------------------------------------------------------------- source sampling (S3–S5)
struct Sampled { double x, y, z, u, v, w, E; int group; bool rejected; int ring; };   // ring = the PSR the particle is from

Sampled sample_history(const Psl &psl, const Beam &beam, const uint64_t *off, uint64_t seed, uint64_t h) {
  const PsrParams &p = psl.p;
  size_t G = psl.groups.size(), g = 0;
  while (g + 1 < G && !(h >= off[g] && h < off[g + 1])) ++g;       // group of history h
  const Group &grp = psl.groups[g];
  Stream st{seed, h, 0, 0};
  uint32_t blk0[4], blk1[4];
  st.next_block(blk0); st.next_block(blk1);           // blocks 0 and 1 of track 0 are the source draws
  uint32_t x0 = blk0[0], x1 = blk0[1], x2 = blk0[2], x3 = blk0[3], y0 = blk1[0], y1 = blk1[1];
  // 1. let through the alias table
  uint64_t m = (uint64_t)x0 * (uint64_t)grp.thresh.size();
  uint32_t col = (uint32_t)(m >> 32), frac = (uint32_t)m;
  uint32_t let = frac < grp.thresh[col] ? col : grp.alias[col];
  // 2. position, uniform in the let's area
  double px, py, pz = p.z_phsp;
  if (psl.mode == 0) {
    double r0 = grp.ring[let] * p.ring_width, r1 = (grp.ring[let] + 1) * p.ring_width;
    double r = std::sqrt(r0 * r0 + U_co(x1) * (r1 * r1 - r0 * r0));
    double th = 2.0 * PI * ((double)grp.sector[let] + U_co(x2)) / psl.n_sectors;
    px = r * std::cos(th); py = r * std::sin(th);
  } else {                                   // square let (Xbin, Ybin): uniform in x and in y (:82)
    px = psl.grid_x0 + ((double)grp.ring[let] + U_co(x1)) * psl.let_size;
    py = psl.grid_x0 + ((double)grp.sector[let] + U_co(x2)) * psl.let_size;
  }
  // the PSR this particle is from: a sector let lies in one ring; a square let's particle belongs to
  // the ring its position falls in
  int psr_ring = psl.mode == 0 ? (int)grp.ring[let] : std::min(p.n_ring - 1, (int)std::floor(std::sqrt(px * px + py * py) / p.ring_width));
  // 3. energy, uniform in the bin
  double E = (p.e_min + grp.ebin * p.e_bin_width) + U_oc(x3) * p.e_bin_width;
  int s = grp.stype;
  if (psl.dir[s].K > 0) {
    // S4 / S5: direction from the Gaussian mixture of the PSR the position falls in
    const Psl::DirModel &dm = psl.dir[s];
    uint32_t y2 = blk1[2];
    double r = std::sqrt(px * px + py * py);
    int i = (int)std::floor(r / p.ring_width); if (i > p.n_ring - 1) i = p.n_ring - 1;      // ring index of the position (:94)
    size_t base = ((size_t)grp.ebin * p.n_ring + i) * dm.K;
    double t = U_co(y0); int k = 0;
    while (k < dm.K - 1 && t >= dm.P[base + k]) ++k;                                         // sequential search of P_{i,k} (:107)
    double rho_n = std::sqrt(-2.0 * std::log(U_oc(y1))), psi = 2.0 * PI * U_co(y2);
    double alpha = dm.mu[base + k] + dm.sa[base + k] * rho_n * std::cos(psi);                // Eq. 6 / Eq. 7
    double beta = dm.sb[base + k] * rho_n * std::sin(psi);
    const double LIM = 1.5;                                                                  // keep tan() finite
    alpha = std::fmax(-LIM, std::fmin(LIM, alpha)); beta = std::fmax(-LIM, std::fmin(LIM, beta));
    double ul = std::tan(alpha), vl = std::tan(beta), wl = 1.0;                              // alpha = atan(u/w), beta = atan(v/w)
    double nl = std::sqrt(ul * ul + vl * vl + wl * wl); ul /= nl; vl /= nl; wl /= nl;
    double th = std::atan2(py, px);                                                          // local (u radial) -> global (:92)
    double dx = ul * std::cos(th) - vl * std::sin(th), dy = ul * std::sin(th) + vl * std::cos(th), dz = wl;
    // jaw rejection on the jaws' upper surfaces (:103): the ray from p along d at each jaw plane
    const Jaws &j = psl.jaws;
    double xj = px + dx / dz * (j.z_jx - pz), yj = py + dy / dz * (j.z_jy - pz);
    bool pass = xj >= j.x1 * j.z_jx / j.sad && xj <= j.x2 * j.z_jx / j.sad &&
                yj >= j.y1 * j.z_jy / j.sad && yj <= j.y2 * j.z_jy / j.sad;
    const double *R = beam.R;
    double bx = px, by = py, bz = pz - beam.sad;
    Sampled o;
    o.x = beam.iso[0] + R[0] * bx + R[1] * by + R[2] * bz;
    o.y = beam.iso[1] + R[3] * bx + R[4] * by + R[5] * bz;
    o.z = beam.iso[2] + R[6] * bx + R[7] * by + R[8] * bz;
    o.u = R[0] * dx + R[1] * dy + R[2] * dz;
    o.v = R[3] * dx + R[4] * dy + R[5] * dz;
    o.w = R[6] * dx + R[7] * dy + R[8] * dz;
    o.E = E; o.group = (int)g; o.rejected = !pass; o.ring = psr_ring;
    return o;
  }
  // 4. source point from the 2-D Gaussian of the sub-source (Eq. 4)
  double rho = p.sigma_src[s] * std::sqrt(-2.0 * std::log(U_oc(y0)));
  double psi = 2.0 * PI * U_co(y1);
  double qx = rho * std::cos(psi), qy = rho * std::sin(psi), qz = p.z_src[s];
  // 5. direction = unit vector source point → phase-space point (Eq. 5)
  double dx = px - qx, dy = py - qy, dz = pz - qz;
  double L = std::sqrt(dx * dx + dy * dy + dz * dz);
  dx /= L; dy /= L; dz /= L;
  // 6. jaw test on the jaws' planes (thin absorbers)
  const Jaws &j = psl.jaws;
  double tx = (j.z_jx - qz) / (pz - qz), ty = (j.z_jy - qz) / (pz - qz);
  double xj = qx + (px - qx) * tx, yj = qy + (py - qy) * ty;
  bool pass = xj >= j.x1 * j.z_jx / j.sad && xj <= j.x2 * j.z_jx / j.sad &&
              yj >= j.y1 * j.z_jy / j.sad && yj <= j.y2 * j.z_jy / j.sad;
  // 7. beam set-up
  const double *R = beam.R;
  double bx = px, by = py, bz = pz - beam.sad;
  Sampled o;
  o.x = beam.iso[0] + R[0] * bx + R[1] * by + R[2] * bz;
  o.y = beam.iso[1] + R[3] * bx + R[4] * by + R[5] * bz;
  o.z = beam.iso[2] + R[6] * bx + R[7] * by + R[8] * bz;
  o.u = R[0] * dx + R[1] * dy + R[2] * dz;
  o.v = R[3] * dx + R[4] * dy + R[5] * dz;
  o.w = R[6] * dx + R[7] * dy + R[8] * dz;
  o.E = E; o.group = (int)g; o.rejected = !pass; o.ring = psr_ring;
  return o;
}

// ---------------------------------------------------------------- physics (P1–P9)
double sigma_kn(double E) {   // Klein–Nishina total cross-section per electron, cm^2
  double a = E / ME, L = std::log(1.0 + 2.0 * a);
  return 2.0 * PI * RE2 * ((1.0 + a) / (a * a) * (2.0 * (1.0 + a) / (1.0 + 2.0 * a) - L / a) + L / (2.0 * a) -
                           (1.0 + 3.0 * a) / ((1.0 + 2.0 * a) * (1.0 + 2.0 * a)));
}
void mu_over_rho(int m, double E, double out[3]) {   // Compton, photo, pair; cm^2/g
  out[0] = NE[m] * sigma_kn(E);
  out[1] = CPHOTO[m] / (E * E * E);
  double l = E > E_PAIR ? std::log(E / E_PAIR) : 0.0;
  out[2] = PPAIR[m] * l * l;
}
double stopping(int m, double T) { return SSCALE[m] * (1.52 + 0.25 / T + 0.078 * T); }   // MeV cm^2/g

void rotate(double d[3], double ct, double st, double phi) {
  double cp = std::cos(phi), sp = std::sin(phi), nx, ny, nz;
  double s2 = d[0] * d[0] + d[1] * d[1];               // = 1 - d_z^2 for a unit vector (P8)
  if (s2 > 1e-20) {
    double s = std::sqrt(s2);
    nx = d[0] * ct + st * (d[0] * d[2] * cp - d[1] * sp) / s;
    ny = d[1] * ct + st * (d[1] * d[2] * cp + d[0] * sp) / s;
    nz = d[2] * ct - s * st * cp;
  } else {
    nx = st * cp; ny = st * sp; nz = (d[2] > 0 ? ct : -ct);
  }
  double n = std::sqrt(nx * nx + ny * ny + nz * nz);
  d[0] = nx / n; d[1] = ny / n; d[2] = nz / n;
}

// Kahn's rejection for Klein–Nishina; returns eta = E/E'.  One block per trial: words 0, 1, 2 = r1, r2, r3; word 3
// of the ACCEPTED trial is returned in `w_phi` (the caller's azimuth draw).
double kahn(double alpha, Stream &st, uint32_t &w_phi, uint64_t *n_trials = nullptr, int *branch = nullptr) {
  for (;;) {
    uint32_t w[4]; st.next_block(w);
    if (n_trials) ++*n_trials;
    double r1 = U_co(w[0]), r2 = U_co(w[1]), r3 = U_co(w[2]);
    w_phi = w[3];
    if (r1 <= (2.0 * alpha + 1.0) / (2.0 * alpha + 9.0)) {
      double eta = 1.0 + 2.0 * alpha * r2;
      if (r3 <= 4.0 * (1.0 / eta - 1.0 / (eta * eta))) { if (branch) *branch = 0; return eta; }
    } else {
      double eta = (2.0 * alpha + 1.0) / (1.0 + 2.0 * alpha * r2);
      double ct = 1.0 - (eta - 1.0) / alpha;
      if (r3 <= 0.5 * (ct * ct + 1.0 / eta)) { if (branch) *branch = 1; return eta; }
    }
  }
}

struct Track { double pos[3], dir[3], E; int type; uint64_t h; uint32_t track, nblk, nchild; };   // nblk: first stream block of the track's transport
struct Event { uint32_t track; char code; double pos[3], dir[3], E, aux; };

struct Ctx {
  Phantom ph; uint64_t seed; int flags; double fE;
  int64_t *acc; Result *res; i128 ledger[4]; double rhomax[3];
  std::vector<Track> stack; uint64_t fp; std::vector<Event> *trace;
  Fnv *cur = nullptr;                 // fingerprint of the track being transported (FLAG_FP_VOXELS: deposits hash their voxel into it)

  void init(const Phantom &p) {
    ph = p; ledger[0] = ledger[1] = ledger[2] = ledger[3] = 0; trace = nullptr; fE = FE_DEFAULT;
    rhomax[0] = rhomax[1] = rhomax[2] = 0;
    size_t n = (size_t)p.nx * p.ny * p.nz;
    for (size_t v = 0; v < n; ++v) { int m = p.material[v]; if (p.density[v] > rhomax[m]) rhomax[m] = p.density[v]; }
  }
  static int64_t quanta(double E) { return (int64_t)std::llrint(E * FIX); }
  void ev(const Track &t, char code, double aux = 0) {
    if (trace) { Event e; e.track = t.track; e.code = code; std::memcpy(e.pos, t.pos, 24); std::memcpy(e.dir, t.dir, 24); e.E = t.E; e.aux = aux; trace->push_back(e); }
  }
  bool locate(const double pos[3], int ijk[3]) const {
    double fi = std::floor((pos[0] - ph.ox) / ph.dx), fj = std::floor((pos[1] - ph.oy) / ph.dy), fk = std::floor((pos[2] - ph.oz) / ph.dz);
    if (!(fi >= 0 && fi < ph.nx && fj >= 0 && fj < ph.ny && fk >= 0 && fk < ph.nz)) return false;
    ijk[0] = (int)fi; ijk[1] = (int)fj; ijk[2] = (int)fk; return true;
  }
  size_t vox(const int ijk[3]) const { return ((size_t)ijk[2] * ph.ny + ijk[1]) * ph.nx + ijk[0]; }
  // Commissioning tally: com_index[v] = 0 (voxel not needed) or 1 + row; com_dose[col * com_rows + row]
  // with col = the PSR unit of the history (all descendants inherit it).
  const int32_t *com_index = nullptr; int64_t *com_dose = nullptr; int64_t com_rows = 0; uint32_t com_col = 0;
  void deposit(size_t v, double dE, uint32_t tag = 0) {
    int64_t q = quanta(dE); acc[v] += q; ledger[1] += q; ++res->n_deposits;
    if ((flags & FLAG_FP_VOXELS) && cur) cur->u32((uint32_t)v | tag);
    if (com_index && com_index[v] > 0) com_dose[(size_t)com_col * com_rows + (com_index[v] - 1)] += q;
  }
  void escape(double E) { ledger[2] += quanta(E); }
  // Ray/box entry: false = the track misses the phantom.
  bool enter(Track &t, int ijk[3]) const {
    const double lo[3] = {ph.ox, ph.oy, ph.oz};
    const double hi[3] = {ph.ox + ph.nx * ph.dx, ph.oy + ph.ny * ph.dy, ph.oz + ph.nz * ph.dz};
    double tmin = -std::numeric_limits<double>::infinity(), tmax = std::numeric_limits<double>::infinity();
    for (int a = 0; a < 3; ++a) {
      if (t.dir[a] == 0.0) { if (t.pos[a] < lo[a] || t.pos[a] >= hi[a]) return false; continue; }
      double t1 = (lo[a] - t.pos[a]) / t.dir[a], t2 = (hi[a] - t.pos[a]) / t.dir[a];
      if (t1 > t2) { double s = t1; t1 = t2; t2 = s; }
      if (t1 > tmin) tmin = t1; if (t2 < tmax) tmax = t2;
    }
    if (tmin > tmax || tmax <= 0.0) return false;
    double s = (tmin > 0.0 ? tmin : 0.0) + EPS_B;
    for (int a = 0; a < 3; ++a) t.pos[a] += s * t.dir[a];
    return locate(t.pos, ijk);
  }
  double mu_max(double E) const {
    double best = 0;
    for (int m = 0; m < 3; ++m) { double c[3]; mu_over_rho(m, E, c); double v = rhomax[m] * (c[0] + c[1] + c[2]); if (v > best) best = v; }
    return best;
  }
  void charged_secondary(const Track &parent, const double dir[3], double T, uint32_t slot, size_t v) {
    if (T >= ECUT && !(flags & FLAG_ELECTRONS_LOCAL)) {
      Track c; std::memcpy(c.pos, parent.pos, 24); std::memcpy(c.dir, dir, 24); c.E = T; c.type = 1; c.h = parent.h;
      c.track = child_track(parent.track, parent.nchild, slot); c.nblk = 0; c.nchild = 0;
      stack.push_back(c); ++res->n_sec_electrons;
    } else deposit(v, T);
  }

  void photon(Track t) {
    Fnv f; f.u32(t.track); cur = &f;
    Stream st{seed, t.h, t.track, t.nblk};
    int ijk[3]; bool collided = false;
    if (flags & FLAG_TRACE_BIRTH) ev(t, 'B');
    if (!locate(t.pos, ijk) && !enter(t, ijk)) { escape(t.E); f.byte('M'); ev(t, 'M'); ++res->n_missed; fp += f.v; return; }
    for (;;) {
      if (t.E < PCUT) { deposit(vox(ijk), t.E); f.byte('A'); ev(t, 'A'); ++res->n_photon_cutoff; break; }
      double mmax = mu_max(t.E);
      if (!(mmax > 0.0)) { escape(t.E); f.byte('E'); ev(t, 'E'); ++res->n_photon_escape; if (!collided && t.track == 0) ++res->n_uncollided_escape; break; }
      uint32_t wf[4]; st.next_block(wf);               // flight: word 0 = free path, word 1 = choice of interaction
      double s = -std::log(U_oc(wf[0])) / mmax;
      for (int a = 0; a < 3; ++a) t.pos[a] += s * t.dir[a];
      ++res->n_flights;
      if (!locate(t.pos, ijk)) { escape(t.E); f.byte('E'); ev(t, 'E', s); ++res->n_photon_escape; if (!collided && t.track == 0) ++res->n_uncollided_escape; break; }
      size_t v = vox(ijk); double rho = ph.density[v]; int m = ph.material[v];
      double c[3]; mu_over_rho(m, t.E, c);
      double muC = rho * c[0], muT = rho * c[1], muK = rho * c[2];
      double tt = U_co(wf[1]) * mmax;
      if (tt < muC) {                                  // Compton, Klein–Nishina by Kahn
        collided = true; ++res->n_compton; f.byte('C');
        uint32_t w_phi; int branch = 0; double alpha = t.E / ME, eta = kahn(alpha, st, w_phi, &res->n_kahn_trials, &branch);
        if (flags & FLAG_FP_VOXELS) f.u32(st.j | (branch ? 0x80000000u : 0u));
        double k = (eta - 1.0) / alpha, ct = 1.0 - k, sn = std::sqrt(std::fmax(0.0, k * (2.0 - k)));
        double phi = 2.0 * PI * U_co(w_phi);
        double Ep = t.E / eta, T = t.E - Ep, d0[3] = {t.dir[0], t.dir[1], t.dir[2]};
        rotate(t.dir, ct, sn, phi);
        double de[3] = {t.E * d0[0] - Ep * t.dir[0], t.E * d0[1] - Ep * t.dir[1], t.E * d0[2] - Ep * t.dir[2]};
        double n = std::sqrt(de[0] * de[0] + de[1] * de[1] + de[2] * de[2]);
        if (n > 0) { de[0] /= n; de[1] /= n; de[2] /= n; } else { de[0] = d0[0]; de[1] = d0[1]; de[2] = d0[2]; }
        ev(t, 'C', ct);
        charged_secondary(t, de, T, 0, v); ++t.nchild;
        t.E = Ep;
      } else if (tt < muC + muT) {                     // photo-electric: local absorption
        ++res->n_photo; f.byte('P'); ev(t, 'P'); deposit(v, t.E); break;
      } else if (tt < muC + muT + muK) {               // pair production
        ++res->n_pair; f.byte('X'); ev(t, 'X');
        uint32_t wp[4]; st.next_block(wp);             // pair: word 0 = energy split, 1 = cos, 2 = azimuth of the annihilation pair
        double Tsum = t.E - E_PAIR, Tm = U_co(wp[0]) * Tsum, Tp = Tsum - Tm;
        charged_secondary(t, t.dir, Tm, 0, v);
        charged_secondary(t, t.dir, Tp, 1, v);
        double cz = 2.0 * U_co(wp[1]) - 1.0, sz = std::sqrt(std::fmax(0.0, 1.0 - cz * cz)), az = 2.0 * PI * U_co(wp[2]);
        double nrm[3] = {sz * std::cos(az), sz * std::sin(az), cz};
        for (uint32_t slot = 2; slot < 4; ++slot) {
          Track c; std::memcpy(c.pos, t.pos, 24); double sg = slot == 2 ? 1.0 : -1.0;
          for (int a = 0; a < 3; ++a) c.dir[a] = sg * nrm[a];
          c.E = E_ANNIH; c.type = 0; c.h = t.h; c.track = child_track(t.track, t.nchild, slot); c.nblk = 0; c.nchild = 0;
          stack.push_back(c); ++res->n_sec_photons;
        }
        ++t.nchild; break;
      } else { ++res->n_virtual; f.byte('V'); ev(t, 'V'); }
    }
    fp += f.v;
  }

  void electron(Track t) {
    Fnv f; f.u32(t.track); cur = &f;
    Stream st{seed, t.h, t.track, t.nblk};
    ++res->n_electron_tracks;
    int ijk[3]; uint32_t steps = 0;
    if (flags & FLAG_TRACE_BIRTH) ev(t, 'B');
    if (!locate(t.pos, ijk) && !enter(t, ijk)) { escape(t.E); f.u32(0); f.byte('M'); ev(t, 'M'); ++res->n_missed; fp += f.v; return; }
    const double lo[3] = {ph.ox, ph.oy, ph.oz}, dd[3] = {ph.dx, ph.dy, ph.dz};
    // One condensed-history step loses the fraction fE of the energy it starts with (budget); it is cut
    // into sub-steps at voxel faces.  The Gaussian deflection is applied once per condensed step, over
    // the rho*s/X0 accumulated along it (P7).
    double budget = 0, tacc = 0, Tms = t.E; bool fresh = true;
    for (;;) {
      if (fresh) { budget = fE * t.E; Tms = t.E; tacc = 0; fresh = false; }
      size_t v = vox(ijk); double rho = ph.density[v]; int m = ph.material[v];
      double D = stopping(m, t.E) * rho;
      double sE = D > 0 ? budget / D : std::numeric_limits<double>::infinity();
      double sv = std::numeric_limits<double>::infinity();
      for (int a = 0; a < 3; ++a) {
        if (t.dir[a] > 0) sv = std::fmin(sv, (lo[a] + (ijk[a] + 1) * dd[a] - t.pos[a]) / t.dir[a]);
        else if (t.dir[a] < 0) sv = std::fmin(sv, (lo[a] + ijk[a] * dd[a] - t.pos[a]) / t.dir[a]);
      }
      if (sv < 0) sv = 0;
      bool turn = sE <= sv + EPS_B;                       // the sub-step ends the condensed step
      double s = turn ? sE : sv + EPS_B, dT = turn ? budget : D * s;
      ++steps; ++res->n_electron_steps;
      const uint32_t tag = turn ? 0x80000000u : 0u;
      if (t.E - dT <= ECUT) { deposit(v, t.E, tag); ev(t, 'A', s); f.u32(steps); f.byte('A'); break; }
      deposit(v, dT, tag);
      for (int a = 0; a < 3; ++a) t.pos[a] += s * t.dir[a];
      t.E -= dT; budget -= dT; tacc += rho * s / X0[m];
      if (!locate(t.pos, ijk)) { escape(t.E); ev(t, 'E', s); ++res->n_electron_escape; f.u32(steps); f.byte('E'); break; }
      if (turn) {
        double pbeta = Tms * (Tms + 2.0 * ME) / (Tms + ME);
        double th0 = 13.6 / pbeta * std::sqrt(tacc);
        uint32_t wd[4]; st.next_block(wd);             // deflection: word 0 = Gaussian radius, word 1 = azimuth
        double a1 = U_oc(wd[0]), b1 = U_co(wd[1]);
        double th = std::fmin(PI, th0 * std::sqrt(-2.0 * std::log(a1)));
        rotate(t.dir, std::cos(th), std::sin(th), 2.0 * PI * b1);
        fresh = true; ++res->n_deflections;
        ev(t, 'T', s);
      } else ev(t, 'S', s);
    }
    fp += f.v;
  }

  void run_history() {   // drains the stack; order is irrelevant (streams are keyed by track)
    while (!stack.empty()) { Track t = stack.back(); stack.pop_back(); if (t.type == 0) photon(t); else electron(t); }
  }
  void store_ledgers() {
    for (int i = 0; i < 4; ++i) { res->ledger_hi[i] = (int64_t)(ledger[i] >> 64); res->ledger_lo[i] = (uint64_t)ledger[i]; }
  }
};

}  // namespace

// ==================================================================== C API (ctypes; oracle/__init__.py)
extern "C" {

void orc_philox(uint64_t seed, uint64_t h, uint32_t track, uint32_t block, uint32_t *out) { philox_block(seed, h, track, block, out); }
uint32_t orc_child_track(uint32_t parent, uint32_t n, uint32_t c) { return child_track(parent, n, c); }

void *orc_psl_build(const PsrParams *p, const Jaws *j, int32_t n_sectors) { return psl_build(*p, *j, n_sectors); }
// Eq. 6 / Eq. 7 parameters of one sub-source: c, mu, sigma_alpha, sigma_beta as [n_ebin][n_ring][K]; K = 0 switches back.
void orc_psl_set_direction(void *h, int32_t stype, int32_t K, const double *c, const double *mu, const double *sa, const double *sb) {
  Psl &psl = *(Psl *)h; Psl::DirModel &dm = psl.dir[stype];
  dm.K = K; size_t n = (size_t)psl.p.n_ebin * psl.p.n_ring * (K > 0 ? K : 0);
  dm.P.assign(n, 0); dm.mu.assign(mu, mu + n); dm.sa.assign(sa, sa + n); dm.sb.assign(sb, sb + n);
  for (size_t b = 0; b < n; b += K) {
    double tot = 0, run = 0; for (int k = 0; k < K; ++k) tot += c[b + k];
    for (int k = 0; k < K; ++k) { run += c[b + k]; dm.P[b + k] = run / tot; }
  }
}
void *orc_psl_build_grid(const PsrParams *p, const Jaws *j, double let_size) { return psl_build_grid(*p, *j, let_size); }
int32_t orc_psl_grid_n(const void *h) { return ((const Psl *)h)->n_xy; }
double orc_psl_grid_x0(const void *h) { return ((const Psl *)h)->grid_x0; }
void orc_psl_free(void *h) { delete (Psl *)h; }
int32_t orc_psl_n_groups(const void *h) { return (int32_t)((const Psl *)h)->groups.size(); }
int64_t orc_psl_group_size(const void *h, int32_t g) { return (int64_t)((const Psl *)h)->groups[g].ring.size(); }
double orc_psl_group_weight(const void *h, int32_t g) { return ((const Psl *)h)->groups[g].W; }
void orc_psl_group_get(const void *h, int32_t g, uint16_t *ring, uint16_t *sector, uint32_t *thresh, uint32_t *alias) {
  const Group &G = ((const Psl *)h)->groups[g];
  for (size_t i = 0; i < G.ring.size(); ++i) { ring[i] = G.ring[i]; sector[i] = G.sector[i]; thresh[i] = G.thresh[i]; alias[i] = G.alias[i]; }
}
void orc_psl_rect(const void *h, double *out) { std::memcpy(out, ((const Psl *)h)->rect, sizeof(double) * 12); }
void orc_allocate(const void *h, uint64_t N, uint64_t *off) { allocate(*(const Psl *)h, N, off); }

// out: count rows of 8 doubles: x, y, z, u, v, w, E, status (group, or -(group)-1 if jaw-rejected)
void orc_sample(const void *h, const Beam *beam, uint64_t N, uint64_t seed, uint64_t first, uint64_t count, double *out) {
  const Psl &psl = *(const Psl *)h;
  std::vector<uint64_t> off(psl.groups.size() + 1); allocate(psl, N, off.data());
  for (uint64_t i = 0; i < count; ++i) {
    Sampled s = sample_history(psl, *beam, off.data(), seed, first + i);
    double *o = out + 8 * i;
    o[0] = s.x; o[1] = s.y; o[2] = s.z; o[3] = s.u; o[4] = s.v; o[5] = s.w; o[6] = s.E;
    o[7] = s.rejected ? -(double)s.group - 1.0 : (double)s.group;
  }
}

// One history of an N-history allocation: source sampling, then its whole shower.  Returns the history's fingerprint.
static uint64_t run_one_history(const Psl &psl, const Beam &beam, const uint64_t *off, uint64_t seed, uint64_t hh, Ctx &c, Result *res) {
  Sampled s = sample_history(psl, beam, off, seed, hh);
  int stype = psl.groups[s.group].stype;
  ++res->n_hist[stype];
  c.ledger[0] += Ctx::quanta(s.E);
  c.fp = 0;
  if (s.rejected) {
    c.ledger[3] += Ctx::quanta(s.E); ++res->n_jaw_rejected;
    Fnv f; f.u32(0); f.byte('J'); c.fp += f.v;
  } else {
    Track t; t.pos[0] = s.x; t.pos[1] = s.y; t.pos[2] = s.z; t.dir[0] = s.u; t.dir[1] = s.v; t.dir[2] = s.w; t.E = s.E;
    t.type = psl.p.particle_type[stype]; t.h = hh; t.track = 0; t.nblk = 2; t.nchild = 0;
    c.stack.push_back(t); c.run_history();
  }
  return c.fp;
}

// Full path for histories [h_begin, h_end) of an N-history allocation.  acc: int64[nvox], ADDED to.
// fingerprints: u64[h_end-h_begin] or NULL, ADDED to.
int32_t orc_dose(const void *h, const Phantom *ph, const Beam *beam, uint64_t N, uint64_t seed, uint64_t h_begin,
                 uint64_t h_end, int32_t flags, int64_t *acc, Result *res, uint64_t *fingerprints) {
  const Psl &psl = *(const Psl *)h;
  std::memset(res, 0, sizeof(Result));
  Ctx c; c.init(*ph); c.seed = seed; c.flags = flags; c.acc = acc; c.res = res;
  std::vector<uint64_t> off(psl.groups.size() + 1); allocate(psl, N, off.data());
  for (uint64_t hh = h_begin; hh < h_end; ++hh) {
    uint64_t fp = run_one_history(psl, *beam, off.data(), seed, hh, c, res);
    if (fingerprints) fingerprints[hh - h_begin] += fp;
  }
  c.store_ledgers();
  return 0;
}

// The same for a LIST of history ids (tests: the tally of a chosen set of histories).  fingerprints: u64[count] or NULL.
int32_t orc_dose_list(const void *h, const Phantom *ph, const Beam *beam, uint64_t N, uint64_t seed, const uint64_t *ids,
                      uint64_t count, int32_t flags, int64_t *acc, Result *res, uint64_t *fingerprints) {
  const Psl &psl = *(const Psl *)h;
  std::memset(res, 0, sizeof(Result));
  Ctx c; c.init(*ph); c.seed = seed; c.flags = flags; c.acc = acc; c.res = res;
  std::vector<uint64_t> off(psl.groups.size() + 1); allocate(psl, N, off.data());
  for (uint64_t i = 0; i < count; ++i) {
    uint64_t fp = run_one_history(psl, *beam, off.data(), seed, ids[i], c, res);
    if (fingerprints) fingerprints[i] += fp;
  }
  c.store_ledgers();
  return 0;
}

// Column of the commissioning matrix for a particle of sub-source s, energy bin e, ring r: one per
// photon PSR, one per electron energy bin ("effective electron PSR unit").
uint32_t orc_com_column(int32_t n_ebin, int32_t n_ring, int32_t particle_type, int32_t s, int32_t e, int32_t r) {
  return particle_type == 0 ? (uint32_t)((s * n_ebin + e) * n_ring + r) : (uint32_t)(2 * n_ebin * n_ring + e);
}

// orc_dose with the commissioning tally: com_index int32[nvox], com_dose int64[com_cols * com_rows] (ADDED to).
int32_t orc_dose_com(const void *h, const Phantom *ph, const Beam *beam, uint64_t N, uint64_t seed, uint64_t h_begin,
                     uint64_t h_end, int64_t *acc, Result *res, const int32_t *com_index, int64_t *com_dose, int64_t com_rows) {
  const Psl &psl = *(const Psl *)h;
  std::memset(res, 0, sizeof(Result));
  Ctx c; c.init(*ph); c.seed = seed; c.flags = 0; c.acc = acc; c.res = res;
  c.com_index = com_index; c.com_dose = com_dose; c.com_rows = com_rows;
  std::vector<uint64_t> off(psl.groups.size() + 1); allocate(psl, N, off.data());
  for (uint64_t hh = h_begin; hh < h_end; ++hh) {
    Sampled s = sample_history(psl, *beam, off.data(), seed, hh);
    const Group &g = psl.groups[s.group];
    ++res->n_hist[g.stype];
    c.ledger[0] += Ctx::quanta(s.E);
    if (s.rejected) { c.ledger[3] += Ctx::quanta(s.E); ++res->n_jaw_rejected; continue; }
    c.com_col = orc_com_column(psl.p.n_ebin, psl.p.n_ring, psl.p.particle_type[g.stype], g.stype, g.ebin, s.ring);
    Track t; t.pos[0] = s.x; t.pos[1] = s.y; t.pos[2] = s.z; t.dir[0] = s.u; t.dir[1] = s.v; t.dir[2] = s.w; t.E = s.E;
    t.type = psl.p.particle_type[g.stype]; t.h = hh; t.track = 0; t.nblk = 2; t.nchild = 0;
    c.fp = 0; c.stack.push_back(t); c.run_history();
  }
  c.store_ledgers();
  return 0;
}

// Transport only: particles rows of 8 doubles as produced by orc_sample (status < 0 skipped).
int32_t orc_transport(const Phantom *ph, int32_t type, const double *particles, uint64_t first, uint64_t count,
                      uint64_t seed, int32_t flags, double fE, int64_t *acc, Result *res, uint64_t *fingerprints) {
  std::memset(res, 0, sizeof(Result));
  Ctx c; c.init(*ph); c.seed = seed; c.flags = flags; c.acc = acc; c.res = res; if (fE > 0) c.fE = fE;
  for (uint64_t i = 0; i < count; ++i) {
    const double *p = particles + 8 * i;
    if (p[7] < 0) continue;
    Track t; for (int a = 0; a < 3; ++a) { t.pos[a] = p[a]; t.dir[a] = p[3 + a]; }
    t.E = p[6]; t.type = type; t.h = first + i; t.track = 0; t.nblk = 2; t.nchild = 0;
    c.ledger[0] += Ctx::quanta(t.E); c.fp = 0;
    c.stack.push_back(t); c.run_history();
    if (fingerprints) fingerprints[i] += c.fp;
  }
  c.store_ledgers();
  return 0;
}

// Event trace of one particle (and all its descendants).  events: rows of 10 doubles
// (track, code, x, y, z, u, v, w, E, aux); returns the number of events (may exceed max_events).
int32_t orc_trace(const Phantom *ph, int32_t type, const double *particle, uint64_t history, uint64_t seed,
                  int32_t flags, double fE, double *events, int32_t max_events) {
  std::vector<int64_t> acc((size_t)ph->nx * ph->ny * ph->nz, 0); Result res; std::memset(&res, 0, sizeof res);
  std::vector<Event> tr;
  Ctx c; c.init(*ph); c.seed = seed; c.flags = flags; c.acc = acc.data(); c.res = &res; c.trace = &tr; if (fE > 0) c.fE = fE;
  Track t; for (int a = 0; a < 3; ++a) { t.pos[a] = particle[a]; t.dir[a] = particle[3 + a]; }
  t.E = particle[6]; t.type = type; t.h = history; t.track = 0; t.nblk = 2; t.nchild = 0;
  c.fp = 0; c.stack.push_back(t); c.run_history();
  for (size_t i = 0; i < tr.size() && (int32_t)i < max_events; ++i) {
    double *o = events + 10 * i; const Event &e = tr[i];
    o[0] = e.track; o[1] = e.code; o[2] = e.pos[0]; o[3] = e.pos[1]; o[4] = e.pos[2];
    o[5] = e.dir[0]; o[6] = e.dir[1]; o[7] = e.dir[2]; o[8] = e.E; o[9] = e.aux;
  }
  return (int32_t)tr.size();
}

// Component probes for the pins.
double orc_sigma_kn(double E) { return sigma_kn(E); }
void orc_mu_over_rho(int32_t m, double E, double *out3) { mu_over_rho(m, E, out3); }
double orc_stopping(int32_t m, double T) { return stopping(m, T); }
// Kahn sampling at fixed E: stream of history first+i, track 0, starting at block 0; one block per trial.
void orc_kahn(double E, uint64_t seed, uint64_t first, uint64_t count, double *cos_out, double *eprime_out) {
  for (uint64_t i = 0; i < count; ++i) {
    Stream st{seed, first + i, 0, 0};
    uint32_t w_phi;
    double alpha = E / ME, eta = kahn(alpha, st, w_phi);
    cos_out[i] = 1.0 - (eta - 1.0) / alpha; eprime_out[i] = E / eta;
  }
}
void orc_rotate(double *d, double ct, double st, double phi) { rotate(d, ct, st, phi); }

// dose[v] = acc[v] 2^-32 / (rho_v V N), MeV/g per history; 0 where rho = 0.
void orc_finalise(const Phantom *ph, const int64_t *acc, uint64_t N, double *dose) {
  size_t n = (size_t)ph->nx * ph->ny * ph->nz; double V = ph->dx * ph->dy * ph->dz;
  for (size_t v = 0; v < n; ++v) { double rho = ph->density[v]; dose[v] = rho > 0 ? (double)acc[v] / FIX / (rho * V * (double)N) : 0.0; }
}

}  // extern "C"
