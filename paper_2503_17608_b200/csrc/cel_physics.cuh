// cel_physics.cuh — the action kernels of one step iteration (docs/PHYSICS_SPEC.md S1, P3i + P3m + P4):
//   k_photoelectric  [PE range]            S8 photoelectric
//   k_pair           [PAIR range]          S8 Bethe-Heitler pair
//   k_annihilation   [ANNIH range]         S8 annihilation at rest
//   k_photon         [COMPTON+MOVE_G]      S8 Compton, then S5 photon move (a Compton survivor moves in the same iteration)
//   k_charged        [MOVE_C+BREMS]        S8 bremsstrahlung, then S7 charged move (step limit, helix, CSDA loss, MSC)
// Each kernel runs only over its action's contiguous range of the sorted index array; in the masked
// modes (`none`, `by particle`) it runs over the whole / the particle's range and the dense key byte masks
// non-participants before any state is read. Scoring (P4, S10) happens here, at the point where the
// deposit is known: warp-aggregated u64 fixed-point atomics, so no deposit is ever staged in HBM.
// One thread per sorted index tid; slot = state_indices[tid], identity in mode `none`.
#pragma once
#include "cel_device.cuh"

namespace cel {

constexpr int kBlock = 256;  // threads per block of the action kernels

// ---------------------------------------------------------------- warp-aggregated integer adds (S10)
// Lanes of the currently converged set that hit the same cell are combined first (__match_any_sync), one leader
// issues the atomic. Integer addition is associative, so the result does not depend on the grouping, on thread
// order or on the sort mode (BASELINE.json config 3: tallies bit-identical across sort modes).
__device__ __forceinline__ void warp_aggregated_add64(unsigned long long* base, unsigned long long cell, unsigned long long value) {
  const unsigned active = __activemask();
  const unsigned peers = __match_any_sync(active, cell);
  const int lane = threadIdx.x & 31;
  const int leader = __ffs(peers) - 1;
  unsigned long long sum = 0;
  unsigned rem = peers;
  while (rem) {  // every lane of a peer group walks the same mask
    const int src = __ffs(rem) - 1;
    sum += __shfl_sync(peers, value, src);
    rem &= rem - 1;
  }
  if (lane == leader) atomicAdd(base + cell, sum);
}
// the per-tile counters of the bookkeeping kernels (vacancies created, secondaries staged): lanes of the converged set
// that hit the same tile are combined first, so a warp issues one atomic per distinct tile. value is 0..3: the peer sums
// are formed from two ballots. (Per-GROUP counters kept by the action kernels as well were tried and dropped: at 2^20
// slots that is 32 addresses for the whole GPU, and same-address atomics serialise in L2 — +7 us per iteration at the
// shower maximum.)
__device__ __forceinline__ void warp_aggregated_add32(uint32_t* tile_cnt, uint32_t tile, uint32_t value) {
  const unsigned active = __activemask();
  const unsigned b0 = __ballot_sync(active, value & 1u), b1 = __ballot_sync(active, value & 2u);
  const unsigned peers = __match_any_sync(active, tile);
  if ((peers & ((1u << (threadIdx.x & 31)) - 1u)) == 0) atomicAdd(tile_cnt + tile, (uint32_t)__popc(peers & b0) + 2u * (uint32_t)__popc(peers & b1));
}

// Hit records (option "hits"): the lanes of the converged set that have a hit reserve their places in the
// device batch buffer with ONE atomic (warp-aggregated), then write their 16-byte records; overflow is a sticky error.
__device__ __forceinline__ void append_hit(const DeviceState& D, bool has, uint32_t event, int bin, unsigned long long q) {
  const unsigned active = __activemask();
  const unsigned m = __ballot_sync(active, has);
  if (m == 0) return;
  const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
  unsigned long long base = 0;
  if (lane == leader) base = atomicAdd(&D.ctl->n_hits, (unsigned long long)__popc(m));
  base = __shfl_sync(active, base, leader);
  if (has) {
    const unsigned long long at = base + (unsigned long long)__popc(m & ((1u << lane) - 1u));
    if (at < D.hit_capacity) {
      asm volatile("st.global.v2.b64 [%0], {%1,%2};" ::"l"(D.hits + at), "l"((unsigned long long)event | ((unsigned long long)(uint32_t)bin << 32)), "l"(q) : "memory");
    } else {
      D.ctl->error = -10;   // CEL_ERR_HIT_OVERFLOW (sticky)
    }
  }
}

// P4 (S10): q = llrint(e * 2^36) added to tally[event][bin]; bin = bin of the volume at the start of the iteration
__device__ __forceinline__ void score(const DeviceState& D, uint32_t event, int vol0, double edep, double eesc) {
  const unsigned long long row = (unsigned long long)event * (unsigned long long)(D.P.n_bins + 1);
  const long long q_dep = quantise(edep);
  int bin = -1;
  if (q_dep != 0) {
    bin = __ldg(D.P.vol_bin + vol0);
    if (bin >= 0) warp_aggregated_add64(D.tally, row + (unsigned long long)bin, (unsigned long long)q_dep);
  }
  const long long q_esc = quantise(eesc);
  if (q_esc != 0) warp_aggregated_add64(D.tally, row + (unsigned long long)D.P.n_bins, (unsigned long long)q_esc);
  // S10: a single deposit of 2^63 quanta = 2^27 MeV or more (the conversion saturates to the largest integer), a negative
  // or a non-finite one (the most negative integer): sticky CEL_ERR_TALLY_OVERFLOW. q + 1 has its top bit set in all of them.
  if ((((unsigned long long)q_dep + 1ull) | ((unsigned long long)q_esc + 1ull)) >> 63) D.ctl->error = -5;
  if (D.hits != nullptr) {   // the same integers, as records for the host (a measurement / application mode)
    append_hit(D, q_dep != 0 && bin >= 0, event, bin, (unsigned long long)q_dep);
    append_hit(D, q_esc != 0, event, D.P.n_bins, (unsigned long long)q_esc);
  }
}

// ---------------------------------------------------------------- the registers of one track
struct Track {
  RecA a;                 // x, y, z, energy
  double dx, dy, dz;
  int ptype, vol, surf;
  uint32_t nsteps, event;
};

__device__ __forceinline__ void stage_secondary(const DeviceState& D, uint32_t slot, int j, const Track& t, double energy,
                                                double dx, double dy, double dz, int ptype) {
  RecA a = t.a; a.energy = energy;
  RecB b; b.dx = dx; b.dy = dy; b.dz = dz;
  b.meta = make_meta(ptype == P_GAMMA ? A_MOVE_G : A_MOVE_C, ptype, t.vol, t.surf, 0, t.event);
  store_a(D.secA + 2ull * slot + j, a);
  store_b(D.secB + 2ull * slot + j, b);
}

// S9-R (sort mode 4): the slot its interaction vacates takes the interaction's first secondary in place —
// the track P1 would have made of that initializer (parent's event, position, vol, surf; nsteps = 0). Returns its action.
__device__ __forceinline__ int become_secondary(Track& t, double energy, double dx, double dy, double dz, int ptype) {
  t.a.energy = energy; t.dx = dx; t.dy = dy; t.dz = dz; t.ptype = ptype; t.nsteps = 0;
  return ptype == P_GAMMA ? A_MOVE_G : A_MOVE_C;
}

// a charged track whose kinetic energy dropped below the cut (its energy is already in edep): returns the new action
__device__ __forceinline__ int stop_charged(const Params& P, int ptype, double& edep) {
  if (ptype == P_POSITRON) {
    if (P.enable_annihilation) return A_ANNIH;
    edep += 2.0 * kElectronMass;
  }
  return A_VACANT;
}

// common epilogue: score, write the slot back, keep the dense key byte and the per-tile counters (vacancies created,
// secondaries staged) that the scans of the next P5/P1 start from
__device__ __forceinline__ void finish(const DeviceState& D, uint32_t slot, uint32_t k_iter, const Track& t, int action, int vol0, double edep,
                                       double eesc, int nsec, bool write_a) {
  score(D, t.event, vol0, edep, eesc);
  // a non-finite energy or position must not go on (grid_locate would send a NaN to cell 0): sticky CEL_ERR_NONFINITE.
  // Exponent-field tests (a few integer operations; a non-finite direction shows in the position one step later).
  if ((((__double2hiint(t.a.energy) & 0x7ff00000) == 0x7ff00000) | ((__double2hiint((t.a.x + t.a.y) + t.a.z) & 0x7ff00000) == 0x7ff00000))) D.ctl->error = -6;
  const uint32_t tile = slot >> D.tile_shift;
  if (D.reuse && action == A_VACANT && nsec >= 1) {
    // S9-R, the general case (the interaction epilogues handle theirs without staging): the slot ends the iteration
    // VACANT with a staged secondary — a Compton / bremsstrahlung survivor whose move then escaped or stopped. Its
    // first staged secondary (written above by this thread) becomes the slot's track, as P1 would have made it.
    const RecA sa = load_a(D.secA + 2ull * slot);
    const RecB sb = load_b(D.secB + 2ull * slot);
    if (nsec == 2) { store_a(D.secA + 2ull * slot, load_a(D.secA + 2ull * slot + 1)); store_b(D.secB + 2ull * slot, load_b(D.secB + 2ull * slot + 1)); }
    store_a(D.stA + slot, sa);
    store_b(D.stB + slot, sb);
    D.akey[slot] = make_key(meta_action(sb.meta), meta_ptype(sb.meta));
    if (nsec == 2) { D.nsec[slot] = 1; warp_aggregated_add32(D.tile_sec, tile, 1u); }
    return;
  }
  RecB b; b.dx = t.dx; b.dy = t.dy; b.dz = t.dz;
  b.meta = make_meta(action, t.ptype, t.vol, t.surf, t.nsteps, t.event);
  if (write_a) store_a(D.stA + slot, t.a);
  store_b(D.stB + slot, b);
  D.akey[slot] = make_key(action, t.ptype);
  if (nsec) {
    D.nsec[slot] = (uint8_t)nsec;
    warp_aggregated_add32(D.tile_sec, tile, (uint32_t)nsec);
  }
  if (action == A_VACANT) {   // into the buffer the fill of iteration k+1 reads (parity (k+1)&1)
    const uint32_t q = D.vac_buf_override ? (uint32_t)(D.vac_buf_override - 1) : (k_iter & 1u) ^ 1u;
    warp_aggregated_add32(D.tile_vac + (size_t)q * D.n_tiles, tile, 1u);
  }
}

__device__ __forceinline__ Track unpack(const RecA& a, const RecB& b) {
  Track t;
  t.a = a; t.dx = b.dx; t.dy = b.dy; t.dz = b.dz;
  t.ptype = meta_ptype(b.meta); t.vol = meta_vol(b.meta); t.surf = meta_surf(b.meta);
  t.nsteps = meta_nsteps(b.meta); t.event = meta_event(b.meta);
  return t;
}

// ================================================================ P3i: pure interactions (the slot is vacated)
// Loop over the kernel's index range with a grid-stride loop; `slot` is the gathered slot index.
#define CEL_FOR_RANGE(RANGE_ID, KERNEL_ID)                                                                  \
  pdl_prologue();                                                                                           \
  const Control* ctl = D.ctl;                                                                               \
  /* (a sticky error also stops the action kernels: a bad device-resident primary must not be stepped) */  \
  const uint32_t finished_ = ctl->finished | (uint32_t)ctl->error;   /* the loads are issued together: one round trip */ \
  const uint32_t rb0_ = ctl->rb[RANGE_ID][0], re0_ = ctl->re[RANGE_ID][0];                                  \
  const uint32_t rb1_ = ctl->rb[RANGE_ID][1], re1_ = ctl->re[RANGE_ID][1];                                  \
  const uint32_t k_iter = ctl->iter;                                                                        \
  if (finished_) return;                                                                                    \
  const TraceScope<KERNEL_ID, TRACE> trace(D, k_iter);                                                      \
  const Params& P = D.P;                                                                                    \
  (void)k_iter; (void)P;                                                                                    \
  /* the kernel's (up to) two index ranges walked as one virtual range with a grid-stride loop */         \
  const uint32_t n0_ = re0_ - rb0_, n_ = n0_ + (re1_ - rb1_);                                               \
  for (uint32_t i_ = blockIdx.x * blockDim.x + threadIdx.x, tid = i_ < n0_ ? rb0_ + i_ : rb1_ + (i_ - n0_); i_ < n_; \
       i_ += gridDim.x * blockDim.x, tid = i_ < n0_ ? rb0_ + i_ : rb1_ + (i_ - n0_))

// Sorted by action a thread walks its kernel's ranges with a grid stride: the slot of its NEXT index is read together with
// the current one, and that slot's two records are prefetched into L1 once the current records have arrived, so that the
// index -> record round trips of all but a thread's first track overlap the arithmetic of the track before.
#define CEL_NEXT_SLOT()                                                                                      \
  uint32_t next_slot_ = 0xffffffffu;                                                                         \
  if (D.sort_mode == 1) {                                                                                    \
    const uint32_t in_ = i_ + gridDim.x * blockDim.x;                                                        \
    if (in_ < n_) next_slot_ = D.indices[in_ < n0_ ? rb0_ + in_ : rb1_ + (in_ - n0_)];                        \
  }
#define CEL_PREFETCH_NEXT()                                                                                  \
  if (next_slot_ != 0xffffffffu) {                                                                           \
    asm volatile("prefetch.global.L1 [%0];" ::"l"(D.stB + next_slot_));                                      \
    asm volatile("prefetch.global.L1 [%0];" ::"l"(D.stA + next_slot_));                                      \
  }

__device__ __forceinline__ uint32_t slot_of(const DeviceState& D, uint32_t tid) { return (D.sort_mode == 1 || D.sort_mode == 2) ? D.indices[tid] : tid; }

// S8 photoelectric: the photon's energy goes to an electron along d (or is deposited when electrons are local)
__device__ __forceinline__ void do_photoelectric(const DeviceState& D, uint32_t slot, uint32_t k_iter, const RecA& a, const RecB& b) {
  Track t = unpack(a, b);
  double edep = 0.0;
  int nsec = 0, action = A_VACANT;
  if (D.P.electrons_local) edep += t.a.energy;
  else if (D.reuse) action = become_secondary(t, t.a.energy, t.dx, t.dy, t.dz, P_ELECTRON);   // only the meta word changes
  else stage_secondary(D, slot, nsec++, t, t.a.energy, t.dx, t.dy, t.dz, P_ELECTRON);
  finish(D, slot, k_iter, t, action, t.vol, edep, 0.0, nsec, false);
}
template <bool TRACE>
__global__ void __launch_bounds__(kBlock) k_photoelectric(DeviceState D) {
  CEL_FOR_RANGE(R_PE, K_PE) {
    const uint32_t slot = slot_of(D, tid);
    if (D.sort_mode != 1 && (D.akey[slot] & 0xf) != A_PE) continue;
    const RecB b = load_b(D.stB + slot);
    const RecA a = load_a(D.stA + slot);   // issued with b: one round trip, not two
    if (meta_action(b.meta) != A_PE) continue;
    do_photoelectric(D, slot, k_iter, a, b);
  }
}

// S8 pair: uniform sharing of E - 2 m_e, both collinear; staging order e-, e+
__device__ __forceinline__ void do_pair(const DeviceState& D, uint32_t slot, uint32_t k_iter, const RecA& a, const RecB& b) {
  const Params& P = D.P;
  Track t = unpack(a, b);
  double edep = 0.0;
  int nsec = 0;
  double xi0, xi1;
  draw_pair(P, slot, k_iter, PH_INTERACT, 0, xi0, xi1);
  const double Tav = t.a.energy - 2.0 * kElectronMass;
  const double Tm = xi0 * Tav;
  const double Tp = Tav - Tm;
  if (D.reuse) {   // S9-R: the first staged secondary (e-, or e+ when the e- is below the cut) takes the slot
    int action;
    if (Tm >= P.cut) { stage_secondary(D, slot, nsec++, t, Tp, t.dx, t.dy, t.dz, P_POSITRON); action = become_secondary(t, Tm, t.dx, t.dy, t.dz, P_ELECTRON); }
    else { edep += Tm; action = become_secondary(t, Tp, t.dx, t.dy, t.dz, P_POSITRON); }
    finish(D, slot, k_iter, t, action, t.vol, edep, 0.0, nsec, true);
    return;
  }
  if (Tm >= P.cut) stage_secondary(D, slot, nsec++, t, Tm, t.dx, t.dy, t.dz, P_ELECTRON);
  else edep += Tm;
  stage_secondary(D, slot, nsec++, t, Tp, t.dx, t.dy, t.dz, P_POSITRON);
  finish(D, slot, k_iter, t, A_VACANT, t.vol, edep, 0.0, nsec, false);
}
template <bool TRACE>
__global__ void __launch_bounds__(kBlock) k_pair(DeviceState D) {
  CEL_FOR_RANGE(R_PAIR, K_PAIR) {
    const uint32_t slot = slot_of(D, tid);
    if (D.sort_mode != 1 && (D.akey[slot] & 0xf) != A_PAIR) continue;
    const RecB b = load_b(D.stB + slot);
    const RecA a = load_a(D.stA + slot);   // issued with b: one round trip, not two
    if (meta_action(b.meta) != A_PAIR) continue;
    do_pair(D, slot, k_iter, a, b);
  }
}

// S8 annihilation at rest: two photons of m_e, back to back, isotropic
__device__ __forceinline__ void do_annihilation(const DeviceState& D, uint32_t slot, uint32_t k_iter, const RecA& a, const RecB& b) {
  Track t = unpack(a, b);
  double xi0, xi1;
  draw_pair(D.P, slot, k_iter, PH_INTERACT, 0, xi0, xi1);
  const double cost = 2.0 * xi0 - 1.0;
  const double sint = sqrt(1.0 - cost * cost);
  double sp, cp;
  sincospi(2.0 * xi1, &sp, &cp);
  const double ux = sint * cp, uy = sint * sp, uz = cost;
  if (D.reuse) {   // S9-R: photon (m_e, u) takes the slot, photon (m_e, -u) is pushed
    stage_secondary(D, slot, 0, t, kElectronMass, -ux, -uy, -uz, P_GAMMA);
    const int action = become_secondary(t, kElectronMass, ux, uy, uz, P_GAMMA);
    finish(D, slot, k_iter, t, action, t.vol, 0.0, 0.0, 1, true);
    return;
  }
  stage_secondary(D, slot, 0, t, kElectronMass, ux, uy, uz, P_GAMMA);
  stage_secondary(D, slot, 1, t, kElectronMass, -ux, -uy, -uz, P_GAMMA);
  finish(D, slot, k_iter, t, A_VACANT, t.vol, 0.0, 0.0, 2, false);
}
template <bool TRACE>
__global__ void __launch_bounds__(kBlock) k_annihilation(DeviceState D) {
  CEL_FOR_RANGE(R_ANNIH, K_ANNIH) {
    const uint32_t slot = slot_of(D, tid);
    if (D.sort_mode != 1 && (D.akey[slot] & 0xf) != A_ANNIH) continue;
    const RecB b = load_b(D.stB + slot);
    const RecA a = load_a(D.stA + slot);   // issued with b: one round trip, not two
    if (meta_action(b.meta) != A_ANNIH) continue;
    do_annihilation(D, slot, k_iter, a, b);
  }
}

// ================================================================ photons: Compton (S8) then move (S5)
// S8 Compton: Klein-Nishina epsilon-mixture rejection; returns the slot's action: MOVE_G (the photon goes on and moves
// in this iteration), VACANT (it fell below the cut), or MOVE_C (S9-R: it fell below the cut and its electron took the slot)
__device__ __forceinline__ int compton(const DeviceState& D, uint32_t slot, uint32_t k_iter, Track& t, double& edep, int& nsec) {
  const Params& P = D.P;
  const double E = t.a.energy;
  const double k = E / kElectronMass;
  const double e0 = 1.0 / (1.0 + 2.0 * k);
  const double a1 = -log(e0);
  const double a2 = (1.0 - e0 * e0) / 2.0;
  double eps, tt, sin2, xphi;
  for (uint32_t trial = 0;; ++trial) {
    double xa, xb, xc;
    draw_pair(P, slot, k_iter, PH_INTERACT, 2 * trial, xa, xb);
    draw_pair(P, slot, k_iter, PH_INTERACT, 2 * trial + 1, xc, xphi);
    if (xa * (a1 + a2) < a1) eps = exp(-a1 * xb);
    else eps = sqrt(e0 * e0 + (1.0 - e0 * e0) * xb);
    tt = (1.0 - eps) / (k * eps);
    sin2 = tt * (2.0 - tt);
    if (xc <= 1.0 - eps * sin2 / (1.0 + eps * eps) || trial >= 65535u) break;
  }
  const double cost = 1.0 - tt;
  const double sint = sqrt(sin2 > 0.0 ? sin2 : 0.0);
  const double E1 = eps * E;
  double d1x = t.dx, d1y = t.dy, d1z = t.dz;
  rotate_dir(d1x, d1y, d1z, cost, sint, 2.0 * xphi);
  const double Te = E - E1;
  if (P.electrons_local || Te < P.cut) {
    edep += Te;
  } else {
    double ex = E * t.dx - E1 * d1x, ey = E * t.dy - E1 * d1y, ez = E * t.dz - E1 * d1z;
    const double n = sqrt(ex * ex + ey * ey + ez * ez);
    if (n > 0.0) { ex /= n; ey /= n; ez /= n; } else { ex = t.dx; ey = t.dy; ez = t.dz; }
    if (D.reuse && E1 < P.cut) { edep += E1; return become_secondary(t, Te, ex, ey, ez, P_ELECTRON); }
    stage_secondary(D, slot, nsec++, t, Te, ex, ey, ez, P_ELECTRON);
  }
  if (E1 < P.cut) { edep += E1; return A_VACANT; }
  t.a.energy = E1; t.dx = d1x; t.dy = d1y; t.dz = d1z;
  return A_MOVE_G;
}

// S5 photon move: sampled free path vs distance to boundary; returns the next action
template <int GEOM>
__device__ __forceinline__ int move_photon(const DeviceState& D, uint32_t slot, uint32_t k_iter, Track& t, double& eesc) {
  const Params& P = D.P;
  const int vol0 = t.vol;
  const int mat = __ldg(P.vol_material + t.vol);
  double sPE = 0.0, sPair = 0.0, sC = 0.0;
  if (mat >= 0) {
    const GridPos g = grid_locate(P, t.a.energy);
    const double2* xs = reinterpret_cast<const double2*>(P.photon_xs + (size_t)mat * kGrid + g.j);  // nodes j, j+1: 64 B
    const double2 n0a = __ldg(xs), n0b = __ldg(xs + 1), n1a = __ldg(xs + 2), n1b = __ldg(xs + 3);
    sC = lerp_node(n0a.x, n1a.x, g.f);
    sPE = lerp_node(n0a.y, n1a.y, g.f);
    sPair = lerp_node(n0b.x, n1b.x, g.f);
  }
  const double stot = (sPE + sPair) + sC;
  double xi0, xi1;
  draw_pair(P, slot, k_iter, PH_STEP, 0, xi0, xi1);
  const double s_d = (stot > 0.0) ? -log(xi0) / stot : CEL_INF;
  const double x = xi1 * stot;
  const int process = (x < sPE) ? A_PE : ((x < sPE + sPair) ? A_PAIR : A_COMPTON);
  int which;
  const double s_b = distance_to_boundary<GEOM>(P, t.a.x, t.a.y, t.a.z, t.dx, t.dy, t.dz, t.vol, t.surf, s_d, which);
  if (t.nsteps < 65535u) t.nsteps += 1;
  if (s_d < s_b) {
    t.a.x += s_d * t.dx; t.a.y += s_d * t.dy; t.a.z += s_d * t.dz;
    t.surf = -1;
    return process;
  }
  t.a.x += s_b * t.dx; t.a.y += s_b * t.dy; t.a.z += s_b * t.dz;
  const bool escaped = cross_boundary<GEOM>(P, t.a.z, t.dz, t.vol, t.surf, which);
  if (escaped) {
    eesc += t.a.energy;
    if (t.vol < 0 || t.vol > 254) t.vol = vol0;
    return A_VACANT;
  }
  return A_MOVE_G;
}

// act = COMPTON: interact, then (if the photon survives) move; act = MOVE_G: move
template <int GEOM>
__device__ __forceinline__ void do_photon(const DeviceState& D, uint32_t slot, uint32_t k_iter, const RecA& a, const RecB& b, int act) {
  Track t = unpack(a, b);
  const int vol0 = t.vol;
  double edep = 0.0, eesc = 0.0;
  int nsec = 0;
  int action = A_MOVE_G;
  if (act == A_COMPTON) action = compton(D, slot, k_iter, t, edep, nsec);
  if (action == A_MOVE_G) action = move_photon<GEOM>(D, slot, k_iter, t, eesc);
  finish(D, slot, k_iter, t, action, vol0, edep, eesc, nsec, true);
}
// (four blocks per SM = 64 registers: measured 1-3 % faster than the 80 the compiler takes unasked)
template <int GEOM, bool TRACE>
__global__ void __launch_bounds__(kBlock, 4) k_photon(DeviceState D) {
  CEL_FOR_RANGE(R_PHOTON, K_PHOTON) {
    const uint32_t slot = slot_of(D, tid);
    CEL_NEXT_SLOT()
    if (D.sort_mode != 1) { const int ak = D.akey[slot] & 0xf; if (ak != A_COMPTON && ak != A_MOVE_G) continue; }
    const RecB b = load_b(D.stB + slot);
    const RecA a = load_a(D.stA + slot);   // issued with b: one round trip, not two
    const int act = meta_action(b.meta);
    CEL_PREFETCH_NEXT()
    if (act != A_COMPTON && act != A_MOVE_G) continue;
    do_photon<GEOM>(D, slot, k_iter, a, b, act);
  }
}

// ================================================================ charged: bremsstrahlung (S8) then move (S7)
// S7: step limit -> linear or helical propagation (<= max_substeps chord substeps) -> CSDA loss -> MSC -> fate.
// The move is written in three parts: step limit (charged_limit), propagation (one straight segment, or chord substeps
// of the helix one at a time), and energy loss + MSC + fate (charged_finish).
struct ChargedStep {      // what the step limit leaves for the parts after the propagation
  double T0, p2, r0, s_phys;
  int mat, j0, vol0;
  bool interaction_wins;
};
struct Prop {             // propagation state of one track in a field (S7.3), advanced one chord substep at a time
  double x, y, z, dx, dy, dz, remaining, travelled, omega, h_max;
  int vol, surf, n;
  int escaped, complete;
};

// S7.1 + S7.2. Returns false if the track stopped at once (S7.1; `action` is then its fate), true if it moves.
__device__ __forceinline__ bool charged_limit(const DeviceState& D, uint32_t slot, uint32_t k_iter, Track& t, double& edep, ChargedStep& c, int& action) {
  const Params& P = D.P;
  c.vol0 = t.vol;
  if (t.nsteps < 65535u) t.nsteps += 1;
  c.T0 = t.a.energy;
  if (c.T0 < P.cut) {  // S7.1
    edep += c.T0;
    t.a.energy = 0.0;
    action = stop_charged(P, t.ptype, edep);
    return false;
  }
  c.mat = __ldg(P.vol_material + t.vol);
  c.p2 = c.T0 * (c.T0 + 2.0 * kElectronMass);   // p^2; beta p = p^2 / (T0 + m_e)
  // S7.2 step limit
  c.r0 = 0.0; c.j0 = 0;
  double s_r = CEL_INF, s_d = CEL_INF;
  if (c.mat >= 0) {
    const GridPos g = grid_locate(P, c.T0);
    c.j0 = g.j;
    const double2* cxs = reinterpret_cast<const double2*>(P.charged_xs + (size_t)c.mat * kGrid + g.j);  // nodes j, j+1
    const double2 n0 = __ldg(cxs);
    const double2 n1 = __ldg(cxs + 1);
    if (P.enable_eloss) {
      c.r0 = lerp_node(n0.y, n1.y, g.f);
      s_r = (c.r0 <= kRhoF) ? c.r0 : fmax(kAlphaR * c.r0, kRhoF);
    }
    const double sb = lerp_node(n0.x, n1.x, g.f);
    double xi0, xi1;
    draw_pair(P, slot, k_iter, PH_STEP, 0, xi0, xi1);
    if (sb > 0.0) s_d = -log(xi0) / sb;
  }
  c.interaction_wins = s_d < s_r;
  c.s_phys = c.interaction_wins ? s_d : s_r;
  return true;
}

// S7.3 without a field: one straight segment
template <int GEOM>
__device__ __forceinline__ void propagate_linear(const Params& P, Track& t, double s_phys, double& travelled, bool& escaped, bool& complete) {
  int which;
  const double s_b = distance_to_boundary<GEOM>(P, t.a.x, t.a.y, t.a.z, t.dx, t.dy, t.dz, t.vol, t.surf, s_phys, which);
  if (s_phys < s_b) {
    t.a.x += s_phys * t.dx; t.a.y += s_phys * t.dy; t.a.z += s_phys * t.dz;
    t.surf = -1; travelled = s_phys; complete = true;
  } else {
    t.a.x += s_b * t.dx; t.a.y += s_b * t.dy; t.a.z += s_b * t.dz;
    travelled = s_b;
    escaped = cross_boundary<GEOM>(P, t.a.z, t.dz, t.vol, t.surf, which);
  }
}

// S7.3 in a field: set up the chord substeps. Returns false if there is nothing to propagate (s_phys = 0).
__device__ __forceinline__ bool prop_begin(const Params& P, const Track& t, const ChargedStep& c, Prop& s) {
  s.x = t.a.x; s.y = t.a.y; s.z = t.a.z; s.dx = t.dx; s.dy = t.dy; s.dz = t.dz;
  s.vol = t.vol; s.surf = t.surf; s.n = 0; s.escaped = 0; s.complete = 0;
  s.travelled = 0.0; s.remaining = c.s_phys;
  const double q = (t.ptype == P_ELECTRON) ? -1.0 : 1.0;
  s.omega = q * kKappa * P.bmag / sqrt(c.p2);
  s.h_max = fmin(sqrt(8.0 * kDeltaChord / fabs(s.omega)), 0.5 / fabs(s.omega));
  if (!(c.s_phys > 0.0)) { s.complete = 1; return false; }
  return true;
}
// one chord substep (S7.3). Returns true while another substep is due in this iteration (not complete, no boundary met,
// fewer than max_substeps made: otherwise the step is paused, and the remainder re-sampled next iteration).
template <int GEOM>
__device__ __forceinline__ bool helix_substep(const Params& P, Prop& s) {
  double h = fmin(s.remaining, s.h_max);
  const HelixFrame F = helix_frame(P, s.dx, s.dy, s.dz);
  // The chord c = pos(h) - pos is used UN-normalised: the distance to the boundary along it then comes out in units of
  // the chord (f = t / |c| of S7.3 directly), "t <= |c|" is "f <= 1", and the sign tests of the dip rule and of the
  // crossing do not care about the scale — no square root and no three divisions per substep (the same reals as S7.3,
  // rounded differently in the last place)
  double nx, ny, nz, ndx, ndy, ndz, cx, cy, cz, fb;
  int which;
  for (int halvings = 0;; ++halvings) {
    helix_point(P, F, s.x, s.y, s.z, s.omega, h, nx, ny, nz, ndx, ndy, ndz);
    cx = nx - s.x; cy = ny - s.y; cz = nz - s.z;
    fb = distance_to_boundary<GEOM>(P, s.x, s.y, s.z, cx, cy, cz, s.vol, s.surf, 1.0, which);
    // S7.3 dip rule: on a surface with the tangent into the volume but the chord out of it, halve h
    if (fb == 0.0 && halvings < kMaxDipHalvings &&
        tangent_points_inward(P, s.x, s.y, s.dx, s.dy, s.dz, cx, cy, cz, which)) { h *= 0.5; continue; }
    break;
  }
  if (fb <= 1.0) {
    double fx, fy, fz, fdx, fdy, fdz;
    helix_point(P, F, s.x, s.y, s.z, s.omega, fb * h, fx, fy, fz, fdx, fdy, fdz);
    s.x += fb * cx; s.y += fb * cy; s.z += fb * cz;
    normalise3(fdx, fdy, fdz);
    s.dx = fdx; s.dy = fdy; s.dz = fdz;
    s.travelled += fb * h;
    s.escaped = cross_boundary<GEOM>(P, s.z, cz, s.vol, s.surf, which) ? 1 : 0;
    return false;
  }
  normalise3(ndx, ndy, ndz);
  s.x = nx; s.y = ny; s.z = nz;
  s.dx = ndx; s.dy = ndy; s.dz = ndz;
  s.travelled += h;
  s.surf = -1;
  s.remaining -= h;
  s.n += 1;
  if (s.remaining <= 0.0) { s.complete = 1; return false; }
  return s.n < P.max_substeps;
}
__device__ __forceinline__ void prop_end(const Prop& s, const ChargedStep& c, Track& t, double& travelled, bool& escaped, bool& complete) {
  t.a.x = s.x; t.a.y = s.y; t.a.z = s.z; t.dx = s.dx; t.dy = s.dy; t.dz = s.dz; t.vol = s.vol; t.surf = s.surf;
  escaped = s.escaped != 0; complete = s.complete != 0;
  travelled = complete ? c.s_phys : s.travelled;
}

// S7.4 - S7.6: energy loss over the travelled path, multiple scattering, fate. Returns the next action.
__device__ __forceinline__ int charged_finish(const DeviceState& D, uint32_t slot, uint32_t k_iter, Track& t, const ChargedStep& c,
                                              double travelled, bool escaped, bool complete, double& edep, double& eesc) {
  const Params& P = D.P;
  const int ptype = t.ptype;
  // S7.4 energy loss
  double T1 = c.T0;
  if (c.mat >= 0 && P.enable_eloss) {
    const double r1 = c.r0 - travelled;
    T1 = (r1 <= 0.0) ? 0.0 : range_inverse(P, P.range_tab + (size_t)c.mat * kGrid, r1, c.j0);
    if (T1 > c.T0) T1 = c.T0;
    edep += c.T0 - T1;
  }
  // S7.5 multiple scattering
  if (P.enable_msc && !escaped && c.mat >= 0 && travelled > 0.0 && T1 >= P.cut) {
    const double x = travelled * __ldg(&P.mats[c.mat].inv_X0);
    const double theta0 = 13.6 * (c.T0 + kElectronMass) / c.p2 * sqrt(x) * fmax(0.0, 1.0 + 0.038 * log(x));
    double xm0, xm1;
    draw_pair(P, slot, k_iter, PH_MSC, 0, xm0, xm1);
    const double theta = fmin(theta0 * sqrt(-2.0 * log(xm0)), kPi);
    double st, ct;
    sincos(theta, &st, &ct);
    rotate_dir(t.dx, t.dy, t.dz, ct, st, 2.0 * xm1);
  }
  // S7.6 fate
  const double rest = (ptype == P_POSITRON) ? 2.0 * kElectronMass : 0.0;
  if (escaped) {
    eesc += T1 + rest; t.a.energy = T1;
    if (t.vol < 0 || t.vol > 254) t.vol = c.vol0;
    return A_VACANT;
  }
  if (T1 < P.cut) {
    edep += T1; t.a.energy = 0.0;
    return stop_charged(P, ptype, edep);
  }
  if (t.nsteps >= P.max_steps_per_track) {
    eesc += T1 + rest; t.a.energy = T1;
    return A_VACANT;
  }
  t.a.energy = T1;
  return (c.interaction_wins && complete) ? A_BREMS : A_MOVE_C;
}

// S8 bremsstrahlung (act = BREMS): k log-uniform on [k_c, T], photon collinear. Returns the action after it: MOVE_C (the
// track goes on and moves in this iteration), or its fate if it stopped.
__device__ __forceinline__ int brems(const DeviceState& D, uint32_t slot, uint32_t k_iter, Track& t, double& edep, int& nsec) {
  const Params& P = D.P;
  double xi0, xi1;
  draw_pair(P, slot, k_iter, PH_INTERACT, 0, xi0, xi1);
  const double kph = P.cut * exp(xi0 * log(t.a.energy / P.cut));
  const double T1 = t.a.energy - kph;
  if (T1 < P.cut) {
    edep += T1;
    int action = stop_charged(P, t.ptype, edep);
    if (D.reuse && action == A_VACANT) action = become_secondary(t, kph, t.dx, t.dy, t.dz, P_GAMMA);   // S9-R: the photon takes the slot
    else { stage_secondary(D, slot, nsec++, t, kph, t.dx, t.dy, t.dz, P_GAMMA); t.a.energy = 0.0; }
    return action;
  }
  stage_secondary(D, slot, nsec++, t, kph, t.dx, t.dy, t.dz, P_GAMMA);
  t.a.energy = T1;
  return A_MOVE_C;
}

// act = BREMS: interact, then (unless the track stopped) move; act = MOVE_C: move
template <bool FIELD, int GEOM>
__device__ __forceinline__ void do_charged(const DeviceState& D, uint32_t slot, uint32_t k_iter, const RecA& a, const RecB& b, int act) {
  const Params& P = D.P;
  Track t = unpack(a, b);
  const int vol0 = t.vol;
  double edep = 0.0, eesc = 0.0;
  int nsec = 0;
  int action = A_MOVE_C;
  if (act == A_BREMS) action = brems(D, slot, k_iter, t, edep, nsec);
  if (action == A_MOVE_C) {
    ChargedStep c;
    if (charged_limit(D, slot, k_iter, t, edep, c, action)) {
      double travelled = 0.0;
      bool escaped = false, complete = false;
      if (!FIELD) {
        propagate_linear<GEOM>(P, t, c.s_phys, travelled, escaped, complete);
      } else {
        Prop s;
        if (prop_begin(P, t, c, s)) while (helix_substep<GEOM>(P, s)) {}
        prop_end(s, c, t, travelled, escaped, complete);
      }
      action = charged_finish(D, slot, k_iter, t, c, travelled, escaped, complete, edep, eesc);
    }
  }
  finish(D, slot, k_iter, t, action, vol0, edep, eesc, nsec, true);
}
// (without a field: four blocks per SM = 64 registers, the count the kernel is tuned at — 70+ registers measured 19 % slower;
// with a field: three blocks per SM = 85 registers with ~200 bytes of spills measured 2 % faster than two blocks at 122.
// Tried and dropped for the field kernel: the block parks its tracks' propagation state in shared memory and makes the chord
// substeps in rounds over a compacted queue, so that warps stay full whatever the mix of 1-substep and 10-substep tracks
// (12.7 of 32 lanes are active inside the per-thread loop): bit-identical, 40 % fewer warp instructions in the loop, but
// 22 % SLOWER on config 3 (20.7 vs 16.9 ms) — every warp of the block then waits at the round barriers for the block's
// slowest track, and the kernel is bound by latency, not by issue slots. DESIGN.md section 10.)
template <bool FIELD, int GEOM, bool TRACE>
__global__ void __launch_bounds__(kBlock, FIELD ? 3 : 4) k_charged(DeviceState D) {
  CEL_FOR_RANGE(R_CHARGED, K_CHARGED) {
    const uint32_t slot = slot_of(D, tid);
    CEL_NEXT_SLOT()
    if (D.sort_mode != 1) { const int ak = D.akey[slot] & 0xf; if (ak != A_MOVE_C && ak != A_BREMS) continue; }
    const RecB b = load_b(D.stB + slot);
    const RecA a = load_a(D.stA + slot);   // issued with b: one round trip, not two
    const int act = meta_action(b.meta);
    CEL_PREFETCH_NEXT()
    if (act != A_MOVE_C && act != A_BREMS) continue;
    do_charged<FIELD, GEOM>(D, slot, k_iter, a, b, act);
  }
}

// ================================================================ the three pure interactions in ONE launch (sort by action)
// Photoelectric, pair and annihilation vacate their slot and are cheap; their ranges are usually small. One grid walks
// 256-index chunks of the three ranges (a block runs one action's code per chunk), so the iteration has three
// action launches instead of five: on this GPU every 1184-block launch of an iteration graph costs ~1.5-3 us of
// serialised front-end time, which in the lightly loaded iterations was the critical path (profiles/: timeline).
// At most 48 registers, so nothing is lost in occupancy (unlike k_actions). Bit-identical to the separate kernels.
template <bool TRACE>
__global__ void __launch_bounds__(kBlock) k_discrete(DeviceState D) {
  pdl_prologue();
  const Control* ctl = D.ctl;
  const uint32_t finished_ = ctl->finished | (uint32_t)ctl->error;
  const uint32_t b_an = ctl->rb[R_ANNIH][0], e_an = ctl->re[R_ANNIH][0];
  const uint32_t b_pe = ctl->rb[R_PE][0], e_pe = ctl->re[R_PE][0];
  const uint32_t b_pa = ctl->rb[R_PAIR][0], e_pa = ctl->re[R_PAIR][0];
  const uint32_t k_iter = ctl->iter;
  if (finished_) return;
  const TraceScope<K_DISCRETE, TRACE> trace(D, k_iter);
  const uint32_t n_an = (e_an - b_an + kBlock - 1) / kBlock, n_pe = (e_pe - b_pe + kBlock - 1) / kBlock;
  const uint32_t n_pa = (e_pa - b_pa + kBlock - 1) / kBlock;
  const uint32_t c1 = n_pe, c2 = c1 + n_an, c3 = c2 + n_pa;
  for (uint32_t v = blockIdx.x; v < c3; v += gridDim.x) {   // block-uniform
    uint32_t tid, end; int want;
    if (v < c1) { tid = b_pe + v * kBlock; end = e_pe; want = A_PE; }
    else if (v < c2) { tid = b_an + (v - c1) * kBlock; end = e_an; want = A_ANNIH; }
    else { tid = b_pa + (v - c2) * kBlock; end = e_pa; want = A_PAIR; }
    tid += threadIdx.x;
    if (tid < end) {
      const uint32_t slot = D.indices[tid];
      const RecB b = load_b(D.stB + slot);
      const RecA a = load_a(D.stA + slot);
      if (meta_action(b.meta) == want) {
        if (want == A_PE) do_photoelectric(D, slot, k_iter, a, b);
        else if (want == A_ANNIH) do_annihilation(D, slot, k_iter, a, b);
        else do_pair(D, slot, k_iter, a, b);
      }
    }
  }
}

// The masked modes' form: one pass over the kernel's index range, the key byte picks the three pure interactions. It
// runs BEFORE the two move kernels (a move kernel rewrites key bytes into PE / PAIR / ANNIH, which must not be applied
// in the same iteration), replacing the chains {annihilation -> charged} and {photoelectric -> pair -> photon}.
template <bool TRACE>
__global__ void __launch_bounds__(kBlock) k_discrete_masked(DeviceState D) {
  pdl_prologue();
  const Control* ctl = D.ctl;
  const uint32_t finished_ = ctl->finished | (uint32_t)ctl->error;
  const uint32_t re = D.N;   // (modes none / partition only: every slot, masked by the key byte)
  const uint32_t k_iter = ctl->iter;
  if (finished_) return;
  const TraceScope<K_DISCRETE, TRACE> trace(D, k_iter);
  for (uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x; tid < re; tid += gridDim.x * blockDim.x) {
    const uint32_t slot = slot_of(D, tid);
    const int ak = D.akey[slot] & 0xf;
    if (ak != A_PE && ak != A_PAIR && ak != A_ANNIH) continue;
    const RecB b = load_b(D.stB + slot);
    const RecA a = load_a(D.stA + slot);
    const int act = meta_action(b.meta);
    if (act == A_PE) do_photoelectric(D, slot, k_iter, a, b);
    else if (act == A_PAIR) do_pair(D, slot, k_iter, a, b);
    else if (act == A_ANNIH) do_annihilation(D, slot, k_iter, a, b);
  }
}

}  // namespace cel
