// cel_oracle.cpp — plain, slow, scalar CPU oracle of docs/PHYSICS_SPEC.md.
//
// TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and the
// cpu_baseline / --impl reference legs of bench.py may build, load or call this file.
// It shares no code, header, table or constant generator with the CUDA path in
// paper_2503_17608_b200/csrc/ and neither includes the other.
//
// What it is: the step iteration of arXiv 2503.17608 section 2 plus the
// index reindexing of section 3.1 and the substep cap of section 3.3
// (PAPER.md:57), over an array-of-structs track array, one function per phase, scalar loops
// over slots in ascending order, following docs/PHYSICS_SPEC.md S0-S11 in its order and notation.
// The physics formulas are those the spec freezes from BASELINE.json (north_star, configs).
//
// Pins (tests/test_oracle_pins_*.py, -m "not gpu"): Philox known answers re-derived with Python
// big integers; Thomson limit and quadrature of the KN differential cross-section; the textbook
// non-relativistic and ultra-relativistic limits of the electron stopping power; exp(-mu x)
// attenuation; KN sampler chi-square and moments vs the analytic pdf; CSDA range vs adaptive
// quadrature of 1/S; helix radius p/(|q|B) and circle membership; geometry distances vs
// ray marching; hand-written (vol, surf) crossing sequences in concentric cylinder shells;
// the tally bin of a step = the volume at the START of the iteration (deposit of a crossing /
// escaping step computed from the range table in the test); the looper-cap fate (escape credit
// T, or T + 2 m_e for e+, after exactly max_steps_per_track steps); brems / pair / annihilation /
// Highland distribution checks; per-event energy conservation; init / sort / push vs an
// independent numpy restatement; the partition rule (mode 3) and the parent-slot reuse rule
// (mode 4) hand-worked and restated against mode 1; sort-mode invariance; OpenMP threads do not
// change a bit.
// Parity unpinned (no external truth exists): per-layer shower profiles of the simplified
// physics (configs 2-5) — sanity checks only (shower maximum, containment).
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -std=c++17 -shared -fPIC (see oracle/build.py).

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

// ---------------------------------------------------------------- S0 constants
const double M_EL = 0.51099895;
const double R_E = 2.8179403262e-13;
const double N_AVO = 6.02214076e23;
const double ALPHA_FS = 7.2973525693e-3;
const double KAPPA = 2.99792458;
const double ALPHA_R = 0.2;
const double RHO_F = 0.01;
const double DELTA_CHORD = 1e-3;
const int MAX_DIP_HALVINGS = 30;   // S7.3 dip rule
const double PI = 3.14159265358979323846;
const double INF = std::numeric_limits<double>::infinity();
const double TALLY_SCALE = 68719476736.0;  // 2^36

enum Action { PE = 0, PAIR = 1, COMPTON = 2, MOVE_G = 3, MOVE_C = 4, BREMS = 5, ANNIH = 6, VACANT = 7 };
enum PType { GAMMA = 0, ELECTRON = 1, POSITRON = 2 };
enum Phase { PH_INTERACT = 0, PH_STEP = 1, PH_MSC = 2 };
enum { TAB_COMPTON = 0, TAB_PE = 1, TAB_PAIR = 2, TAB_BREMS = 3, TAB_RANGE = 4, N_TAB = 5 };
const int N_GRID = 577;

}  // namespace

// ---------------------------------------------------------------- plain C structs of the oracle's own ABI
extern "C" {
struct OrcMaterial { double density, Z, A; };
struct OrcGeometry {
  int kind;  // 0 slab, 1 cylinder
  int n_vol;
  const double* bounds;     // n_vol + 1
  const int* vol_material;  // n_vol, -1 = vacuum
  const int* vol_bin;       // n_vol, -1 = not scored
  double half_x, half_y, half_z;
  double field[3];
};
struct OrcPhysics {
  uint64_t seed;
  double cut;
  int enable_pair, enable_brems, enable_msc, enable_eloss, enable_annihilation;
  int electrons_local;
  int max_substeps;
  uint32_t max_steps_per_track;
  uint64_t init_capacity;
};
struct OrcPrimary { uint32_t event; int ptype; double energy; double pos[3]; double dir[3]; };
struct OrcTrack {
  double pos[3]; double dir[3]; double energy;
  uint32_t event; uint32_t nsteps; int vol; int surf; int ptype; int action;
};
}

namespace {

// ---------------------------------------------------------------- S3 Philox4x32-10
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// draw j of (slot, iteration k, phase)
double uniform_draw(uint64_t seed, uint32_t slot, uint32_t k, uint32_t phase, uint32_t j) {
  uint32_t ctr[4] = {slot, k, phase, j >> 1};
  uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
  uint32_t w[4];
  philox4x32_10(ctr, key, w);
  uint32_t h = j & 1u;
  uint64_t x = ((uint64_t)w[2 * h + 1] << 32) | (uint64_t)w[2 * h];
  return ((double)(x >> 12) + 0.5) * (1.0 / 4503599627370496.0);  // 2^-52
}

// ---------------------------------------------------------------- S0/S4 material data and tables
struct MatData {
  double density, Z, A;
  double n_atom, n_e, I_mev, L_rad, inv_X0;
  double tab[N_TAB][N_GRID];
};

double grid_u0() { return std::log(1e-3); }
double grid_du() { return std::log(10.0) / 64.0; }

double sigma_kn(double E) {
  double k = E / M_EL;
  double l = std::log1p(2.0 * k);
  double t1 = (1.0 + k) / (k * k) * (2.0 * (1.0 + k) / (1.0 + 2.0 * k) - l / k);
  double t2 = l / (2.0 * k);
  double t3 = (1.0 + 3.0 * k) / ((1.0 + 2.0 * k) * (1.0 + 2.0 * k));
  return 2.0 * PI * R_E * R_E * (t1 + t2 - t3);
}

double stopping_power(const MatData& m, double T) {
  double tau = T / M_EL;
  double beta2 = tau * (tau + 2.0) / ((tau + 1.0) * (tau + 1.0));
  double ione = m.I_mev / M_EL;
  double bracket = std::log(tau * tau * (tau + 2.0) / (2.0 * ione * ione)) + 1.0 - beta2 +
                   (tau * tau / 8.0 - (2.0 * tau + 1.0) * std::log(2.0)) / ((tau + 1.0) * (tau + 1.0));
  return 2.0 * PI * R_E * R_E * M_EL * m.n_e / beta2 * bracket;
}

void build_material(MatData& m, const OrcMaterial& in, const OrcPhysics& ph) {
  m.density = in.density; m.Z = in.Z; m.A = in.A;
  m.n_atom = in.density * N_AVO / in.A;
  m.n_e = in.Z * m.n_atom;
  m.I_mev = 16e-6 * std::pow(in.Z, 0.9);
  m.L_rad = std::log(183.0 * std::pow(in.Z, -1.0 / 3.0));
  m.inv_X0 = 4.0 * ALPHA_FS * R_E * R_E * m.n_atom * in.Z * (in.Z + 1.0) * m.L_rad;
  const double n_pb = 11.35 * N_AVO / 207.2;
  const double u0 = grid_u0(), du = grid_du();
  for (int j = 0; j < N_GRID; ++j) {
    double E = std::exp(u0 + j * du);
    m.tab[TAB_COMPTON][j] = m.n_e * sigma_kn(E);
    m.tab[TAB_PE][j] = (m.n_atom / n_pb) * std::pow(in.Z / 82.0, 5.0) * std::pow(E, -3.5);
    double ns = (28.0 / 9.0) * std::log(2.0 * E / M_EL) - 218.0 / 27.0;
    double cs = (28.0 / 9.0) * m.L_rad - 2.0 / 27.0;
    double f = std::fmax(0.0, std::fmin(ns, cs));
    m.tab[TAB_PAIR][j] = ph.enable_pair ? m.n_atom * ALPHA_FS * R_E * R_E * in.Z * (in.Z + 1.0) * f : 0.0;
    m.tab[TAB_BREMS][j] = ph.enable_brems ? std::fmax(0.0, std::log(E / ph.cut)) * m.inv_X0 : 0.0;
  }
  // range by composite Simpson, 64 sub-intervals per cell, integrand e^u / S(e^u)
  m.tab[TAB_RANGE][0] = 0.0;
  for (int j = 1; j < N_GRID; ++j) {
    double a = u0 + (j - 1) * du, b = u0 + j * du;
    const int n = 64;
    double hh = (b - a) / n;
    double sum = 0.0;
    for (int i = 0; i <= n; ++i) {
      double u = a + i * hh;
      double T = std::exp(u);
      double g = T / stopping_power(m, T);
      double wgt = (i == 0 || i == n) ? 1.0 : ((i & 1) ? 4.0 : 2.0);
      sum += wgt * g;
    }
    m.tab[TAB_RANGE][j] = m.tab[TAB_RANGE][j - 1] + sum * hh / 3.0;
  }
}

double table_lookup(const double* y, double E) {
  double t = (std::log(E) - grid_u0()) / grid_du();
  double fl = std::floor(t);
  int j = (fl < 0.0) ? 0 : (fl > 575.0 ? 575 : (int)fl);
  double f = t - (double)j;
  return y[j] + f * (y[j + 1] - y[j]);
}

double range_inverse(const double* R, double r) {
  int lo = 0, hi = N_GRID - 1;  // invariant: R[lo] <= r, answer j in [lo, hi)
  while (hi - lo > 1) {
    int mid = (lo + hi) / 2;
    if (R[mid] <= r) lo = mid; else hi = mid;
  }
  int j = lo;
  double u = grid_u0() + j * grid_du() + grid_du() * (r - R[j]) / (R[j + 1] - R[j]);
  return std::exp(u);
}

// ---------------------------------------------------------------- small vector helpers
void normalise(double v[3]) {
  double n = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
  v[0] /= n; v[1] /= n; v[2] /= n;
}

// S8 rotate(d, theta, phi), taking cos(theta) and sin(theta)
void rotate_dir(const double d[3], double ct, double st, double phi, double out[3]) {
  double sp = std::sin(phi), cp = std::cos(phi);
  double srho = std::sqrt(d[0] * d[0] + d[1] * d[1]);
  if (srho == 0.0) {
    double sg = (d[2] < 0.0) ? -1.0 : 1.0;
    out[0] = st * cp; out[1] = st * sp; out[2] = sg * ct;
  } else {
    out[0] = d[0] * ct + st * (d[0] * d[2] * cp - d[1] * sp) / srho;
    out[1] = d[1] * ct + st * (d[1] * d[2] * cp + d[0] * sp) / srho;
    out[2] = d[2] * ct - srho * st * cp;
  }
  normalise(out);
}

// ---------------------------------------------------------------- S6 geometry
struct Geometry {
  int kind, n_vol;
  std::vector<double> bounds;
  std::vector<int> vol_material, vol_bin;
  double half_x, half_y, half_z;
  double field[3];
};

enum Hit { HIT_NONE = 0, HIT_Z = 1, HIT_X = 2, HIT_Y = 3, HIT_INNER = 4, HIT_OUTER = 5 };

double clamp0(double s) { return s < 0.0 ? 0.0 : s; }

// distance to the boundary of volume `vol` from pos along d; which surface
double distance_to_boundary(const Geometry& g, const double pos[3], const double d[3], int vol, int surf, int* which) {
  if (g.kind == 0) {
    double sz = INF, sx = INF, sy = INF;
    if (d[2] > 0.0) sz = clamp0((g.bounds[vol + 1] - pos[2]) / d[2]);
    else if (d[2] < 0.0) sz = clamp0((g.bounds[vol] - pos[2]) / d[2]);
    if (d[0] > 0.0) sx = clamp0((g.half_x - pos[0]) / d[0]);
    else if (d[0] < 0.0) sx = clamp0((-g.half_x - pos[0]) / d[0]);
    if (d[1] > 0.0) sy = clamp0((g.half_y - pos[1]) / d[1]);
    else if (d[1] < 0.0) sy = clamp0((-g.half_y - pos[1]) / d[1]);
    if (sz <= sx && sz <= sy) { *which = HIT_Z; return sz; }
    if (sx <= sy) { *which = HIT_X; return sx; }
    *which = HIT_Y; return sy;
  }
  // cylinder
  double a = d[0] * d[0] + d[1] * d[1];
  double b = pos[0] * d[0] + pos[1] * d[1];
  double r2 = pos[0] * pos[0] + pos[1] * pos[1];
  double s_in = INF, s_out = INF, s_z = INF;
  if (a != 0.0) {
    {  // outer
      double rho = g.bounds[vol + 1];
      if (surf == vol + 1) {
        s_out = (b >= 0.0) ? 0.0 : -2.0 * b / a;
      } else {
        double c = r2 - rho * rho;
        double D = b * b - a * c;
        if (D < 0.0) D = 0.0;
        s_out = (b > 0.0) ? -c / (b + std::sqrt(D)) : (-b + std::sqrt(D)) / a;
      }
      s_out = clamp0(s_out);
    }
    if (vol > 0) {  // inner
      double rho = g.bounds[vol];
      if (surf == vol) {
        if (b < 0.0) s_in = 0.0;
      } else if (b < 0.0) {
        double c = r2 - rho * rho;
        double D = b * b - a * c;
        if (D > 0.0) s_in = clamp0(c / (-b + std::sqrt(D)));
      }
    }
  }
  if (d[2] > 0.0) s_z = clamp0((g.half_z - pos[2]) / d[2]);
  else if (d[2] < 0.0) s_z = clamp0((-g.half_z - pos[2]) / d[2]);
  if (s_in <= s_out && s_in <= s_z) { *which = HIT_INNER; return s_in; }
  if (s_out <= s_z) { *which = HIT_OUTER; return s_out; }
  *which = HIT_Z; return s_z;
}

// S7.3 dip rule: does the tangent d point INTO the current volume across the surface that the chord ch hits?
// (outward normal of the hit surface: the sign of the chord component for planes, radial for cylinders)
bool tangent_points_inward(const Geometry& g, const double pos[3], const double d[3], const double ch[3], int which) {
  if (g.kind == 0) {
    const int axis = (which == HIT_Z) ? 2 : ((which == HIT_X) ? 0 : 1);
    return d[axis] * ch[axis] < 0.0;
  }
  if (which == HIT_Z) return d[2] * ch[2] < 0.0;
  const double radial = pos[0] * d[0] + pos[1] * d[1];
  return (which == HIT_OUTER) ? (radial < 0.0) : (radial > 0.0);
}

// apply the crossing of surface `which`; returns true if the track escaped
bool cross_boundary(const Geometry& g, double pos[3], const double d[3], int* vol, int* surf, int which) {
  if (g.kind == 0) {
    *surf = -1;
    if (which != HIT_Z) return true;
    if (d[2] > 0.0) { pos[2] = g.bounds[*vol + 1]; *vol += 1; }
    else { pos[2] = g.bounds[*vol]; *vol -= 1; }
    return (*vol < 0 || *vol >= g.n_vol);
  }
  if (which == HIT_Z) { *surf = -1; return true; }
  if (which == HIT_OUTER) { *surf = *vol + 1; *vol += 1; return *vol >= g.n_vol; }
  /* inner */ { *surf = *vol; *vol -= 1; return false; }
}

// ---------------------------------------------------------------- S7.3 helix
// point and direction after arc length h from (pos, d); omega = q kappa |B| / p; bh = unit field
void helix_point(const double pos[3], const double d[3], const double bh[3], double omega, double h,
                 double pos_out[3], double d_out[3]) {
  double dpar = d[0] * bh[0] + d[1] * bh[1] + d[2] * bh[2];
  double dperp[3] = {d[0] - dpar * bh[0], d[1] - dpar * bh[1], d[2] - dpar * bh[2]};
  double w[3] = {d[1] * bh[2] - d[2] * bh[1], d[2] * bh[0] - d[0] * bh[2], d[0] * bh[1] - d[1] * bh[0]};
  double sn = std::sin(omega * h), cs = std::cos(omega * h);
  double sh = std::sin(0.5 * omega * h);
  double A = sn / omega;
  double Bc = 2.0 * sh * sh / omega;
  for (int i = 0; i < 3; ++i) {
    d_out[i] = dpar * bh[i] + cs * dperp[i] + sn * w[i];
    pos_out[i] = pos[i] + h * dpar * bh[i] + A * dperp[i] + Bc * w[i];
  }
}

// ---------------------------------------------------------------- S8 Klein-Nishina sampling
// returns eps; writes tt = (1-eps)/(k eps), sin2 and the index of the accepted trial
double sample_kn(double E, uint64_t seed, uint32_t slot, uint32_t k_iter, double* tt_out, double* sin2_out, uint32_t* trial_out) {
  double k = E / M_EL;
  double e0 = 1.0 / (1.0 + 2.0 * k);
  double a1 = -std::log(e0);
  double a2 = (1.0 - e0 * e0) / 2.0;
  for (uint32_t t = 0;; ++t) {
    double xa = uniform_draw(seed, slot, k_iter, PH_INTERACT, 4 * t);
    double xb = uniform_draw(seed, slot, k_iter, PH_INTERACT, 4 * t + 1);
    double xc = uniform_draw(seed, slot, k_iter, PH_INTERACT, 4 * t + 2);
    double eps;
    if (xa * (a1 + a2) < a1) eps = std::exp(-a1 * xb);
    else eps = std::sqrt(e0 * e0 + (1.0 - e0 * e0) * xb);
    double tt = (1.0 - eps) / (k * eps);
    double sin2 = tt * (2.0 - tt);
    if (xc <= 1.0 - eps * sin2 / (1.0 + eps * eps) || t >= 65535u) {
      *tt_out = tt; *sin2_out = sin2; *trial_out = t;
      return eps;
    }
  }
}

// ---------------------------------------------------------------- the context
struct Initializer {
  double pos[3]; double dir[3]; double energy;
  uint32_t event; int ptype; int vol; int surf;
};

struct Stage {          // per slot, per iteration (S10, S9)
  int64_t q_dep, q_esc; // integer deposits of this iteration
  int bin;              // tally bin of the volume at the start of the iteration
  int nsec;
  Initializer sec[2];
};

struct Oracle {
  Geometry geo;
  std::vector<MatData> mats;
  OrcPhysics phys;
  uint64_t n_slots;
  int sort_mode;
  double bmag; double bh[3];

  std::vector<OrcTrack> tracks;
  std::vector<Stage> stage;
  std::vector<Initializer> init;  // the stack; size() == I
  std::vector<uint32_t> indices;
  uint32_t offsets[9];
  std::vector<uint32_t> counts_log;  // 8 per iteration
  std::vector<uint64_t> tally;       // [n_events][n_bins+1]
  uint32_t n_events; int n_bins;
  uint32_t iter;
  uint64_t track_steps, iterations, secondaries;
  int error;
  int n_threads = 1;   // host threads of the per-slot phases (orc_set_threads)
};

int locate_primary(const Geometry& g, const double pos[3], const double dir[3]) {
  if (g.kind == 0) {
    for (int i = 0; i < g.n_vol; ++i) {
      double lo = g.bounds[i], hi = g.bounds[i + 1];
      if (pos[2] > lo && pos[2] < hi) return i;
      if (pos[2] == lo && dir[2] >= 0.0) return i;
      if (pos[2] == hi && dir[2] < 0.0) return i;
    }
    return -1;
  }
  double r = std::sqrt(pos[0] * pos[0] + pos[1] * pos[1]);
  for (int i = 0; i < g.n_vol; ++i)
    if (r >= g.bounds[i] && r < g.bounds[i + 1]) return i;
  return -1;
}

int64_t quantise(double x) { return (int64_t)std::llrint(x * TALLY_SCALE); }

// ---------------------------------------------------------------- P1 init (S9)
void load_initializer(OrcTrack& t, const Initializer& in) {
  for (int i = 0; i < 3; ++i) { t.pos[i] = in.pos[i]; t.dir[i] = in.dir[i]; }
  t.energy = in.energy; t.event = in.event; t.ptype = in.ptype;
  t.vol = in.vol; t.surf = in.surf; t.nsteps = 0;
  t.action = (in.ptype == GAMMA) ? MOVE_G : MOVE_C;
}

// S9-P (sort mode 3, section 3.2): the initializers popped in this iteration are partitioned by charge and
// assigned to opposite ends of the track array: in pop order, the c-th charged one takes the c-th vacancy counted from
// slot 0 upwards, the g-th neutral one the g-th vacancy counted from slot N-1 downwards.
void phase_init_partition(Oracle& o) {
  uint64_t I = o.init.size();
  std::vector<uint64_t> vacant;
  for (uint64_t s = 0; s < o.n_slots; ++s) if (o.tracks[s].action == VACANT) vacant.push_back(s);
  uint64_t V = vacant.size();
  uint64_t n_take = V < I ? V : I;
  uint64_t c = 0, g = 0;
  for (uint64_t j = 0; j < n_take; ++j) {
    const Initializer& in = o.init[I - 1 - j];
    uint64_t slot = (in.ptype == GAMMA) ? vacant[V - 1 - g++] : vacant[c++];
    load_initializer(o.tracks[slot], in);
  }
  o.init.resize(I - n_take);
}

void phase_init(Oracle& o) {
  if (o.sort_mode == 3) { phase_init_partition(o); return; }
  uint64_t I = o.init.size();
  uint64_t V = 0;
  for (uint64_t s = 0; s < o.n_slots; ++s) V += (o.tracks[s].action == VACANT);
  uint64_t n_take = V < I ? V : I;
  uint64_t rank = 0;
  for (uint64_t s = 0; s < o.n_slots && rank < n_take; ++s) {
    OrcTrack& t = o.tracks[s];
    if (t.action != VACANT) continue;
    const Initializer& in = o.init[I - 1 - rank];
    for (int i = 0; i < 3; ++i) { t.pos[i] = in.pos[i]; t.dir[i] = in.dir[i]; }
    t.energy = in.energy; t.event = in.event; t.ptype = in.ptype;
    t.vol = in.vol; t.surf = in.surf; t.nsteps = 0;
    t.action = (in.ptype == GAMMA) ? MOVE_G : MOVE_C;
    ++rank;
  }
  o.init.resize(I - n_take);
}

// ---------------------------------------------------------------- P2 reindex (S2)
int sort_key(const Oracle& o, const OrcTrack& t) {
  if (o.sort_mode == 1 || o.sort_mode == 4) return t.action;   // mode 4 = by action + parent-slot reuse (S9-R)
  if (o.sort_mode == 2) return t.action == VACANT ? 3 : t.ptype;
  return 0;
}

void phase_reindex(Oracle& o) {
  uint32_t cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (uint64_t s = 0; s < o.n_slots; ++s) cnt[o.tracks[s].action]++;
  for (int a = 0; a < 8; ++a) o.counts_log.push_back(cnt[a]);
  uint64_t alive = o.n_slots - cnt[VACANT];
  o.track_steps += alive;
  if (alive > 0) o.iterations += 1;
  // stable counting sort of slot indices by key
  int n_keys = (o.sort_mode == 1 || o.sort_mode == 4) ? 8 : (o.sort_mode == 2 ? 4 : 1);
  uint32_t kc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (uint64_t s = 0; s < o.n_slots; ++s) kc[sort_key(o, o.tracks[s])]++;
  for (int a = 0; a <= 8; ++a) o.offsets[a] = 0;
  for (int a = 0; a < n_keys; ++a) o.offsets[a + 1] = o.offsets[a] + kc[a];
  for (int a = n_keys; a < 8; ++a) o.offsets[a + 1] = o.offsets[n_keys];
  uint32_t cursor[8];
  for (int a = 0; a < 8; ++a) cursor[a] = o.offsets[a];
  for (uint64_t s = 0; s < o.n_slots; ++s) o.indices[cursor[sort_key(o, o.tracks[s])]++] = (uint32_t)s;
}

// ---------------------------------------------------------------- staging helpers
void stage_secondary(Oracle& o, uint32_t slot, const OrcTrack& parent, int ptype, double energy, const double dir[3]) {
  Stage& st = o.stage[slot];
  Initializer& s = st.sec[st.nsec++];
  for (int i = 0; i < 3; ++i) { s.pos[i] = parent.pos[i]; s.dir[i] = dir[i]; }
  s.energy = energy; s.event = parent.event; s.ptype = ptype; s.vol = parent.vol; s.surf = parent.surf;
}

// a charged track whose kinetic energy dropped below the cut (energy already deposited by the caller)
void stop_charged(Oracle& o, OrcTrack& t, double* edep) {
  t.energy = 0.0;
  if (t.ptype == POSITRON) {
    if (o.phys.enable_annihilation) t.action = ANNIH;
    else { *edep += 2.0 * M_EL; t.action = VACANT; }
  } else {
    t.action = VACANT;
  }
}

// ---------------------------------------------------------------- P3i interactions (S8)
void interact_slot(Oracle& o, uint32_t slot) {
  OrcTrack& t = o.tracks[slot];
  const double cut = o.phys.cut;
  double edep = 0.0;
  switch (t.action) {
    case PE: {
      if (o.phys.electrons_local) edep += t.energy;
      else stage_secondary(o, slot, t, ELECTRON, t.energy, t.dir);
      t.action = VACANT;
    } break;
    case PAIR: {
      double xi0 = uniform_draw(o.phys.seed, slot, o.iter, PH_INTERACT, 0);
      double Tav = t.energy - 2.0 * M_EL;
      double Tm = xi0 * Tav;
      double Tp = Tav - Tm;
      if (Tm >= cut) stage_secondary(o, slot, t, ELECTRON, Tm, t.dir);
      else edep += Tm;
      stage_secondary(o, slot, t, POSITRON, Tp, t.dir);
      t.action = VACANT;
    } break;
    case COMPTON: {
      double tt, sin2; uint32_t trial;
      double E = t.energy;
      double eps = sample_kn(E, o.phys.seed, slot, o.iter, &tt, &sin2, &trial);
      double cost = 1.0 - tt;
      double sint = std::sqrt(sin2 > 0.0 ? sin2 : 0.0);
      double phi = 2.0 * PI * uniform_draw(o.phys.seed, slot, o.iter, PH_INTERACT, 4 * trial + 3);
      double E1 = eps * E;
      double d1[3];
      rotate_dir(t.dir, cost, sint, phi, d1);
      double Te = E - E1;
      double de[3] = {E * t.dir[0] - E1 * d1[0], E * t.dir[1] - E1 * d1[1], E * t.dir[2] - E1 * d1[2]};
      double n = std::sqrt(de[0] * de[0] + de[1] * de[1] + de[2] * de[2]);
      if (n > 0.0) { de[0] /= n; de[1] /= n; de[2] /= n; }
      else { de[0] = t.dir[0]; de[1] = t.dir[1]; de[2] = t.dir[2]; }
      if (o.phys.electrons_local || Te < cut) edep += Te;
      else stage_secondary(o, slot, t, ELECTRON, Te, de);
      if (E1 < cut) { edep += E1; t.action = VACANT; }
      else { t.energy = E1; t.dir[0] = d1[0]; t.dir[1] = d1[1]; t.dir[2] = d1[2]; t.action = MOVE_G; }
    } break;
    case BREMS: {
      double xi0 = uniform_draw(o.phys.seed, slot, o.iter, PH_INTERACT, 0);
      double k = cut * std::exp(xi0 * std::log(t.energy / cut));
      stage_secondary(o, slot, t, GAMMA, k, t.dir);
      double T1 = t.energy - k;
      if (T1 < cut) { edep += T1; stop_charged(o, t, &edep); }
      else { t.energy = T1; t.action = MOVE_C; }
    } break;
    case ANNIH: {
      double xi0 = uniform_draw(o.phys.seed, slot, o.iter, PH_INTERACT, 0);
      double xi1 = uniform_draw(o.phys.seed, slot, o.iter, PH_INTERACT, 1);
      double cost = 2.0 * xi0 - 1.0;
      double sint = std::sqrt(1.0 - cost * cost);
      double phi = 2.0 * PI * xi1;
      double u[3] = {sint * std::cos(phi), sint * std::sin(phi), cost};
      double v[3] = {-u[0], -u[1], -u[2]};
      stage_secondary(o, slot, t, GAMMA, M_EL, u);
      stage_secondary(o, slot, t, GAMMA, M_EL, v);
      t.action = VACANT;
    } break;
    default: return;
  }
  o.stage[slot].q_dep += quantise(edep);
}

// ---------------------------------------------------------------- P3m photon move (S5)
void move_photon(Oracle& o, uint32_t slot) {
  OrcTrack& t = o.tracks[slot];
  double eesc = 0.0;
  int mat = o.geo.vol_material[t.vol];
  double sPE = 0.0, sPair = 0.0, sC = 0.0;
  if (mat >= 0) {
    const MatData& m = o.mats[mat];
    sC = table_lookup(m.tab[TAB_COMPTON], t.energy);
    sPE = table_lookup(m.tab[TAB_PE], t.energy);
    sPair = table_lookup(m.tab[TAB_PAIR], t.energy);
  }
  double stot = (sPE + sPair) + sC;
  double xi0 = uniform_draw(o.phys.seed, slot, o.iter, PH_STEP, 0);
  double xi1 = uniform_draw(o.phys.seed, slot, o.iter, PH_STEP, 1);
  double s_d = (stot > 0.0) ? -std::log(xi0) / stot : INF;
  double x = xi1 * stot;
  int process = (x < sPE) ? PE : ((x < sPE + sPair) ? PAIR : COMPTON);
  int which;
  double s_b = distance_to_boundary(o.geo, t.pos, t.dir, t.vol, t.surf, &which);
  if (t.nsteps < 65535u) t.nsteps += 1;
  if (s_d < s_b) {
    for (int i = 0; i < 3; ++i) t.pos[i] += s_d * t.dir[i];
    t.surf = -1;
    t.action = process;
  } else {
    for (int i = 0; i < 3; ++i) t.pos[i] += s_b * t.dir[i];
    bool escaped = cross_boundary(o.geo, t.pos, t.dir, &t.vol, &t.surf, which);
    if (escaped) { eesc += t.energy; t.action = VACANT; }
    else t.action = MOVE_G;
  }
  o.stage[slot].q_esc += quantise(eesc);
}

// ---------------------------------------------------------------- P3m charged move (S7)
void move_charged(Oracle& o, uint32_t slot) {
  OrcTrack& t = o.tracks[slot];
  const double cut = o.phys.cut;
  double edep = 0.0, eesc = 0.0;
  const double T0 = t.energy;
  if (t.nsteps < 65535u) t.nsteps += 1;
  if (T0 < cut) {  // S7.1
    edep += T0;
    stop_charged(o, t, &edep);
    o.stage[slot].q_dep += quantise(edep);
    return;
  }
  const int mat = o.geo.vol_material[t.vol];
  const double p = std::sqrt(T0 * (T0 + 2.0 * M_EL));
  const double beta = p / (T0 + M_EL);
  // S7.2 step limit
  double r0 = 0.0, s_r = INF, s_d = INF;
  if (mat >= 0) {
    const MatData& m = o.mats[mat];
    if (o.phys.enable_eloss) {
      r0 = table_lookup(m.tab[TAB_RANGE], T0);
      s_r = (r0 <= RHO_F) ? r0 : std::fmax(ALPHA_R * r0, RHO_F);
    }
    double sb = table_lookup(m.tab[TAB_BREMS], T0);
    double xi0 = uniform_draw(o.phys.seed, slot, o.iter, PH_STEP, 0);
    if (sb > 0.0) s_d = -std::log(xi0) / sb;
  }
  const bool interaction_wins = s_d < s_r;
  const double s_phys = interaction_wins ? s_d : s_r;
  // S7.3 propagation
  double travelled = 0.0;
  bool escaped = false, complete = false;
  if (o.bmag == 0.0) {
    int which;
    double s_b = distance_to_boundary(o.geo, t.pos, t.dir, t.vol, t.surf, &which);
    if (s_phys < s_b) {
      for (int i = 0; i < 3; ++i) t.pos[i] += s_phys * t.dir[i];
      t.surf = -1; travelled = s_phys; complete = true;
    } else {
      for (int i = 0; i < 3; ++i) t.pos[i] += s_b * t.dir[i];
      travelled = s_b;
      escaped = cross_boundary(o.geo, t.pos, t.dir, &t.vol, &t.surf, which);
    }
  } else {
    const double q = (t.ptype == ELECTRON) ? -1.0 : 1.0;
    const double omega = q * KAPPA * o.bmag / p;
    const double h_max = std::fmin(std::sqrt(8.0 * DELTA_CHORD / std::fabs(omega)), 0.5 / std::fabs(omega));
    double remaining = s_phys;
    int n = 0;
    if (!(s_phys > 0.0)) complete = true;  // zero-length step (range table gives 0 at the cut)
    while (!complete) {
      if (n == o.phys.max_substeps) break;  // paused
      double h = std::fmin(remaining, h_max);
      double pn[3], dn[3], ch[3], l, tb;
      int which;
      for (int halvings = 0;; ++halvings) {
        helix_point(t.pos, t.dir, o.bh, omega, h, pn, dn);
        double c[3] = {pn[0] - t.pos[0], pn[1] - t.pos[1], pn[2] - t.pos[2]};
        l = std::sqrt(c[0] * c[0] + c[1] * c[1] + c[2] * c[2]);
        for (int i = 0; i < 3; ++i) ch[i] = c[i] / l;
        tb = distance_to_boundary(o.geo, t.pos, ch, t.vol, t.surf, &which);
        // dip rule: on a surface, tangent into the volume but chord out of it -> the helix dips into the volume
        // for less than this h; halve h (not a substep) instead of crossing with zero travel
        if (tb == 0.0 && halvings < MAX_DIP_HALVINGS && tangent_points_inward(o.geo, t.pos, t.dir, ch, which)) { h *= 0.5; continue; }
        break;
      }
      if (tb <= l) {
        double f = tb / l;
        double pf[3], df[3];
        helix_point(t.pos, t.dir, o.bh, omega, f * h, pf, df);
        for (int i = 0; i < 3; ++i) t.pos[i] += tb * ch[i];
        normalise(df);
        for (int i = 0; i < 3; ++i) t.dir[i] = df[i];
        travelled += f * h;
        escaped = cross_boundary(o.geo, t.pos, ch, &t.vol, &t.surf, which);
        break;
      }
      normalise(dn);
      for (int i = 0; i < 3; ++i) { t.pos[i] = pn[i]; t.dir[i] = dn[i]; }
      travelled += h;
      t.surf = -1;
      remaining -= h;
      n += 1;
      if (remaining <= 0.0) { travelled = s_phys; complete = true; break; }
    }
  }
  // S7.4 energy loss
  double T1 = T0;
  if (mat >= 0 && o.phys.enable_eloss) {
    const MatData& m = o.mats[mat];
    double r1 = r0 - travelled;
    T1 = (r1 <= 0.0) ? 0.0 : range_inverse(m.tab[TAB_RANGE], r1);
    if (T1 > T0) T1 = T0;
    edep += T0 - T1;
  }
  // S7.5 multiple scattering
  if (o.phys.enable_msc && !escaped && mat >= 0 && travelled > 0.0 && T1 >= cut) {
    const MatData& m = o.mats[mat];
    double x = travelled * m.inv_X0;
    double theta0 = 13.6 / (beta * p) * std::sqrt(x) * std::fmax(0.0, 1.0 + 0.038 * std::log(x));
    double xm0 = uniform_draw(o.phys.seed, slot, o.iter, PH_MSC, 0);
    double xm1 = uniform_draw(o.phys.seed, slot, o.iter, PH_MSC, 1);
    double theta = std::fmin(theta0 * std::sqrt(-2.0 * std::log(xm0)), PI);
    double phi = 2.0 * PI * xm1;
    double dn[3];
    rotate_dir(t.dir, std::cos(theta), std::sin(theta), phi, dn);
    for (int i = 0; i < 3; ++i) t.dir[i] = dn[i];
  }
  // S7.6 fate
  const double rest = (t.ptype == POSITRON) ? 2.0 * M_EL : 0.0;
  if (escaped) {
    eesc += T1 + rest; t.energy = T1; t.action = VACANT;
  } else if (T1 < cut) {
    edep += T1;
    stop_charged(o, t, &edep);
  } else if (t.nsteps >= o.phys.max_steps_per_track) {
    eesc += T1 + rest; t.energy = T1; t.action = VACANT;
  } else {
    t.energy = T1;
    t.action = (interaction_wins && complete) ? BREMS : MOVE_C;
  }
  o.stage[slot].q_dep += quantise(edep);
  o.stage[slot].q_esc += quantise(eesc);
}

// ---------------------------------------------------------------- P4 score (S10)
void phase_score(Oracle& o) {
  for (uint64_t s = 0; s < o.n_slots; ++s) {
    Stage& st = o.stage[s];
    const OrcTrack& t = o.tracks[s];
    if (st.q_dep != 0 && st.bin >= 0) o.tally[(uint64_t)t.event * (o.n_bins + 1) + st.bin] += (uint64_t)st.q_dep;
    if (st.q_esc != 0) o.tally[(uint64_t)t.event * (o.n_bins + 1) + o.n_bins] += (uint64_t)st.q_esc;
    st.q_dep = 0; st.q_esc = 0;
  }
}

// ---------------------------------------------------------------- P5 push (S9)
// S9-R (sort mode 4, section 3.2): a slot that its interaction vacated in this iteration and that staged
// secondaries takes its first staged secondary in place (exactly the track P1 would make of that initializer); only
// the slot's remaining secondaries are pushed.
void phase_push(Oracle& o) {
  const bool reuse = (o.sort_mode == 4);
  if (reuse) {
    for (uint64_t s = 0; s < o.n_slots; ++s) {
      Stage& st = o.stage[s];
      if (o.tracks[s].action == VACANT && st.nsec >= 1) {
        load_initializer(o.tracks[s], st.sec[0]);
        st.sec[0] = st.sec[1];
        st.nsec -= 1;
      }
    }
  }
  uint64_t S = 0;
  for (uint64_t s = 0; s < o.n_slots; ++s) S += o.stage[s].nsec;
  if (o.init.size() + S > o.phys.init_capacity) { o.error = -4; }
  for (uint64_t s = 0; s < o.n_slots; ++s) {
    Stage& st = o.stage[s];
    for (int j = 0; j < st.nsec; ++j) o.init.push_back(st.sec[j]);
    st.nsec = 0;
  }
  o.secondaries += S;
}

// ---------------------------------------------------------------- one step iteration (S1)
void phases_after_reindex(Oracle& o);

void step_iteration(Oracle& o) {
  phase_init(o);
  phase_reindex(o);
  phases_after_reindex(o);
}

void phases_after_reindex(Oracle& o) {
  // record the tally bin of the volume at the start of the iteration
  for (uint64_t s = 0; s < o.n_slots; ++s) {
    const OrcTrack& t = o.tracks[s];
    o.stage[s].bin = (t.action != VACANT) ? o.geo.vol_bin[t.vol] : -1;
  }
  // P3i: every kernel runs over its range of the sorted index array; the result does not depend on the order.
  // (The two per-slot loops touch only their own slot's track and staging and draw from counter-based streams, so they
  // may run on several host threads — orc_set_threads, OpenMP — with bit-identical results; init, reindex, score and
  // push stay serial. The default is one thread.)
#pragma omp parallel for schedule(static) num_threads(o.n_threads) if (o.n_threads > 1)
  for (uint64_t tid = 0; tid < o.n_slots; ++tid) {
    uint32_t slot = o.indices[tid];
    int a = o.tracks[slot].action;
    if (a == PE || a == PAIR || a == COMPTON || a == BREMS || a == ANNIH) interact_slot(o, slot);
  }
  // P3m
#pragma omp parallel for schedule(dynamic, 256) num_threads(o.n_threads) if (o.n_threads > 1)
  for (uint64_t tid = 0; tid < o.n_slots; ++tid) {
    uint32_t slot = o.indices[tid];
    int a = o.tracks[slot].action;
    // a track set ANNIH-pending or vacated in P3i keeps that action and does not move
    if (a == MOVE_G) move_photon(o, slot);
    else if (a == MOVE_C) move_charged(o, slot);
  }
  phase_score(o);
  phase_push(o);
  o.iter += 1;
}

}  // namespace

// ================================================================ C API (called through ctypes by oracle/oracle.py)
extern "C" {

void* orc_create(const OrcGeometry* g, const OrcMaterial* mats, int n_mats, const OrcPhysics* ph,
                 uint64_t n_slots, int sort_mode) {
  Oracle* o = new Oracle();
  o->geo.kind = g->kind; o->geo.n_vol = g->n_vol;
  o->geo.bounds.assign(g->bounds, g->bounds + g->n_vol + 1);
  o->geo.vol_material.assign(g->vol_material, g->vol_material + g->n_vol);
  o->geo.vol_bin.assign(g->vol_bin, g->vol_bin + g->n_vol);
  o->geo.half_x = g->half_x; o->geo.half_y = g->half_y; o->geo.half_z = g->half_z;
  for (int i = 0; i < 3; ++i) o->geo.field[i] = g->field[i];
  o->phys = *ph;
  if (o->phys.init_capacity == 0) {
    uint64_t c = 8 * n_slots;
    o->phys.init_capacity = c > (1ull << 24) ? c : (1ull << 24);
  }
  o->mats.resize(n_mats);
  for (int i = 0; i < n_mats; ++i) build_material(o->mats[i], mats[i], o->phys);
  o->n_slots = n_slots; o->sort_mode = sort_mode;
  o->bmag = std::sqrt(g->field[0] * g->field[0] + g->field[1] * g->field[1] + g->field[2] * g->field[2]);
  for (int i = 0; i < 3; ++i) o->bh[i] = (o->bmag > 0.0) ? g->field[i] / o->bmag : 0.0;
  int nb = 0;
  for (int i = 0; i < g->n_vol; ++i) if (g->vol_bin[i] + 1 > nb) nb = g->vol_bin[i] + 1;
  o->n_bins = nb;
  o->n_events = 0; o->iter = 0; o->error = 0;
  o->track_steps = o->iterations = o->secondaries = 0;
  return o;
}

void orc_destroy(void* h) { delete (Oracle*)h; }

// host threads used by the per-slot phases P3i / P3m (>= 1); results do not depend on it
void orc_set_threads(void* h, int n) { ((Oracle*)h)->n_threads = n < 1 ? 1 : n; }

int orc_n_bins(void* h) { return ((Oracle*)h)->n_bins; }

// load primaries, reset slots, tallies and counters (S9: primary i -> init[i])
int orc_begin(void* h, const OrcPrimary* prim, uint64_t n, uint32_t n_events) {
  Oracle& o = *(Oracle*)h;
  o.tracks.assign(o.n_slots, OrcTrack());
  for (auto& t : o.tracks) { t.action = VACANT; t.vol = 0; t.surf = -1; }
  o.stage.assign(o.n_slots, Stage());
  for (auto& s : o.stage) { s.q_dep = 0; s.q_esc = 0; s.bin = -1; s.nsec = 0; }
  o.indices.assign(o.n_slots, 0);
  o.init.clear(); o.counts_log.clear();
  o.n_events = n_events;
  o.tally.assign((uint64_t)n_events * (o.n_bins + 1), 0);
  o.iter = 0; o.error = 0; o.track_steps = o.iterations = o.secondaries = 0;
  if (n > o.phys.init_capacity) return -4;
  for (uint64_t i = 0; i < n; ++i) {
    Initializer in;
    for (int c = 0; c < 3; ++c) { in.pos[c] = prim[i].pos[c]; in.dir[c] = prim[i].dir[c]; }
    in.energy = prim[i].energy; in.event = prim[i].event; in.ptype = prim[i].ptype;
    in.vol = locate_primary(o.geo, prim[i].pos, prim[i].dir); in.surf = -1;
    if (in.vol < 0 || prim[i].event >= n_events) return -1;
    o.init.push_back(in);
  }
  return 0;
}

int orc_step(void* h) { Oracle& o = *(Oracle*)h; step_iteration(o); return o.error; }
// the same iteration in three pieces, so that a test can look at the state between phases
void orc_phase_init(void* h) { phase_init(*(Oracle*)h); }
void orc_phase_reindex(void* h) { phase_reindex(*(Oracle*)h); }
int orc_phase_rest(void* h) { Oracle& o = *(Oracle*)h; phases_after_reindex(o); return o.error; }

// run to completion (alive == 0 and I == 0) or max_iter iterations; returns iterations executed or <0
int64_t orc_run(void* h, uint64_t max_iter) {
  Oracle& o = *(Oracle*)h;
  uint64_t n = 0;
  while (n < max_iter) {
    step_iteration(o);
    ++n;
    if (o.error) return o.error;
    uint64_t alive = 0;
    for (uint64_t s = 0; s < o.n_slots; ++s) alive += (o.tracks[s].action != VACANT);
    if (alive == 0 && o.init.empty()) break;
  }
  return (int64_t)n;
}

void orc_read_state(void* h, OrcTrack* out) { Oracle& o = *(Oracle*)h; std::memcpy(out, o.tracks.data(), o.n_slots * sizeof(OrcTrack)); }
void orc_read_indices(void* h, uint32_t* idx, uint32_t* offsets) {
  Oracle& o = *(Oracle*)h;
  std::memcpy(idx, o.indices.data(), o.n_slots * sizeof(uint32_t));
  std::memcpy(offsets, o.offsets, 9 * sizeof(uint32_t));
}
uint64_t orc_n_iterations_logged(void* h) { return ((Oracle*)h)->counts_log.size() / 8; }
void orc_read_counts(void* h, uint32_t* out) { Oracle& o = *(Oracle*)h; std::memcpy(out, o.counts_log.data(), o.counts_log.size() * sizeof(uint32_t)); }
uint64_t orc_n_initializers(void* h) { return ((Oracle*)h)->init.size(); }
// initializers as OrcTrack records (action = -1, nsteps = 0)
void orc_read_initializers(void* h, OrcTrack* out) {
  Oracle& o = *(Oracle*)h;
  for (size_t i = 0; i < o.init.size(); ++i) {
    const Initializer& in = o.init[i];
    for (int c = 0; c < 3; ++c) { out[i].pos[c] = in.pos[c]; out[i].dir[c] = in.dir[c]; }
    out[i].energy = in.energy; out[i].event = in.event; out[i].nsteps = 0;
    out[i].vol = in.vol; out[i].surf = in.surf; out[i].ptype = in.ptype; out[i].action = -1;
  }
}
void orc_read_tallies(void* h, uint64_t* out) { Oracle& o = *(Oracle*)h; std::memcpy(out, o.tally.data(), o.tally.size() * sizeof(uint64_t)); }
void orc_read_counters(void* h, uint64_t* out) {
  Oracle& o = *(Oracle*)h;
  out[0] = o.track_steps; out[1] = o.iterations; out[2] = o.secondaries; out[3] = o.iter;
}

// ---------------------------------------------------------------- unit-level entry points for the pins
void orc_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
double orc_uniform(uint64_t seed, uint32_t slot, uint32_t k, uint32_t phase, uint32_t j) { return uniform_draw(seed, slot, k, phase, j); }
double orc_sigma_kn(double E) { return sigma_kn(E); }
double orc_stopping_power(void* h, int mat, double T) { return stopping_power(((Oracle*)h)->mats[mat], T); }
double orc_inv_X0(void* h, int mat) { return ((Oracle*)h)->mats[mat].inv_X0; }
void orc_table(void* h, int mat, int which, double* out) { std::memcpy(out, ((Oracle*)h)->mats[mat].tab[which], N_GRID * sizeof(double)); }
double orc_lookup(void* h, int mat, int which, double E) { return table_lookup(((Oracle*)h)->mats[mat].tab[which], E); }
double orc_range_inverse(void* h, int mat, double r) { return range_inverse(((Oracle*)h)->mats[mat].tab[TAB_RANGE], r); }
double orc_sample_kn(double E, uint64_t seed, uint32_t slot, uint32_t k, double* tt, double* sin2, uint32_t* trial) {
  return sample_kn(E, seed, slot, k, tt, sin2, trial);
}
void orc_rotate(const double* d, double ct, double st, double phi, double* out) { rotate_dir(d, ct, st, phi, out); }
double orc_distance(void* h, const double* pos, const double* d, int vol, int surf, int* which) {
  return distance_to_boundary(((Oracle*)h)->geo, pos, d, vol, surf, which);
}
void orc_helix_point(const double* pos, const double* d, const double* bh, double omega, double hh, double* pos_out, double* d_out) {
  helix_point(pos, d, bh, omega, hh, pos_out, d_out);
}
int orc_locate(void* h, const double* pos, const double* d) { return locate_primary(((Oracle*)h)->geo, pos, d); }

}  // extern "C"
