// rf_oracle.cpp -- CPU ORACLE for the ROSEFusion hot path (arxiv 2105.05600).  TEST INFRASTRUCTURE.
//
// This file is the plain, slow, obviously-correct restatement of what the CUDA path computes.  It is
// used only by tests/, by __graft_entry__.smoke() and by bench.py's cpu_baseline / --impl reference
// legs.  The product (paper_2105_05600_b200/) never imports, links or executes anything in oracle/,
// and this file shares no code, header, table or helper with the CUDA path.
//
// Citations: "P:L<n>" = /root/reference/PAPER.md line n; "O<n>", "A<n>" = SURVEY.md section 8(c)
// oracle items / readings (restated in DESIGN.md).  Everything is scalar C++ with fp64 arithmetic
// and fp64 accumulation, in the paper's order; no blocking, fusion or reordering.  Where a
// floating-point value decides an integer (valid count of a fitness sample, A26; pixel association
// and band test of the integration, R-I2) the oracle decides in fp64 and FLAGS the inputs whose
// decision a binary32 evaluation could legitimately take the other way ("fragile"); the parity
// gates are exact on everything that is not flagged.
//
// Pins (tests/test_oracle_pins.py): pose algebra P2, back-projection P3, integration P4 (plane,
// sphere, averaging closed forms), trilinear P5 (affine reproduction, scipy cross-check), fitness P6
// (rho = exp(-(a/mu)^2) closed form, 16^3 brute force, identity optimal), swarm update P7 (hand
// case + invariants), whole loop P8 (sanity on synthetic ground truth), ray-cast read-out P9 (plane exact, sphere,
// back face, unobserved gap).
// PARITY UNPINNED against the authors' system (the paper does not determine them; DESIGN.md lists
// each): MovePST frame convention (A2), all integration conventions (A17), F2 normalisation (A6),
// resolution order (A15), the read-out rule (R-R1).  They are pinned only as self-consistent definitions.
//
// Layout conventions: dense volumes are x-fastest, index = x + X*(y + Y*z); tsdf is normalised to
// [-1,1] (distance / trunc); weight is an integer stored as float, 0 = unobserved.  Poses are
// camera-to-world, row-major [R|t] (12 numbers).  K = (fx, fy, cx, cy).
#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>
#include <algorithm>
#include <limits>

extern "C" {

// Constants fixed by the paper.
static const double ORC_TAU = 1.0;      // P:L172  temperature tau = 1
static const double ORC_EPS = 1e-3;     // P:L254  epsilon of Eq. (17)
static const double ORC_BETA = 0.1;     // P:L260  beta of Eq. (18)
static const double ORC_STOP = 1e-6;    // P:L306  change of s_k^* below 1e-6 in all six dims
static const int ORC_EMPTY_STOP = 2;    // P:L306  APS empty for two consecutive steps

struct orc_grid {
  int32_t dims[3];
  float voxel_size;
  float trunc;
  float origin[3];
};

double orc_const(int which) {
  switch (which) {
    case 0: return ORC_TAU;
    case 1: return ORC_EPS;
    case 2: return ORC_BETA;
    case 3: return ORC_STOP;
    case 4: return (double)ORC_EMPTY_STOP;
  }
  return std::numeric_limits<double>::quiet_NaN();
}

// ------------------------------------------------------------------------------------------------
// O2.  Pose from particle (MovePST + RescalePST, Alg. 1 lines 13-14; P:L190 state
// parameterisation (qx,qy,qz,x,y,z); "move and rescale this original PST ... on the fly").
// ------------------------------------------------------------------------------------------------
// Standard rotation matrix of the unit quaternion q = (w, x, y, z).
void orc_quat_to_R(const double q[4], double R[9]) {
  const double w = q[0], x = q[1], y = q[2], z = q[3];
  R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - z * w);     R[2] = 2 * (x * z + y * w);
  R[3] = 2 * (x * y + z * w);     R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - x * w);
  R[6] = 2 * (x * z - y * w);     R[7] = 2 * (y * z + x * w);     R[8] = 1 - 2 * (x * x + y * y);
}

// T_out = Delta(delta) o T_in :  R_out = R(q(delta_q)) * R_in,  t_out = t_in + delta_t   (A2, A3).
// q = (sqrt(max(0, 1 - |delta_q|^2)), delta_q)  -- the particle's rotation block is the imaginary
// part of a unit quaternion; validity guaranteed by |p| <= 1 and r_d <= 1.
void orc_apply_delta(const double T_in[12], const double delta[6], double T_out[12]) {
  double q[4];
  const double s2 = delta[0] * delta[0] + delta[1] * delta[1] + delta[2] * delta[2];
  q[0] = std::sqrt(std::max(0.0, 1.0 - s2));
  q[1] = delta[0]; q[2] = delta[1]; q[3] = delta[2];
  double Rq[9];
  orc_quat_to_R(q, Rq);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      double a = 0;
      for (int k = 0; k < 3; ++k) a += Rq[3 * i + k] * T_in[4 * k + j];
      T_out[4 * i + j] = a;
    }
  for (int i = 0; i < 3; ++i) T_out[4 * i + 3] = T_in[4 * i + 3] + delta[3 + i];
}

// Candidate pose of one particle: delta = r (.) p  (RescalePST on the stored unit-ball template).
void orc_pose_from_particle(const double T_c[12], const double r[6], const float p[6], double T_out[12]) {
  double delta[6];
  for (int d = 0; d < 6; ++d) delta[d] = r[d] * (double)p[d];
  orc_apply_delta(T_c, delta, T_out);
}

// ------------------------------------------------------------------------------------------------
// O3.  Back-projection + stride down-sampling (P:L93 back-projection; P:L294 stride-based
// down-sampling).  Lattice u = floor(s/2) + a*s, v = floor(s/2) + b*s.  Output [M,4] (x,y,z,mask),
// M = number of lattice pixels; pixels with z <= 0 or non-finite get mask 0 (A23).
// ------------------------------------------------------------------------------------------------
int32_t orc_lattice_count(int32_t n, int32_t s) { int32_t h = s / 2; return n > h ? (n - h + s - 1) / s : 0; }

int32_t orc_backproject(const float* depth, int32_t w, int32_t h, const float K[4], int32_t stride,
                        double* pts /* [M,4] */) {
  const double fx = K[0], fy = K[1], cx = K[2], cy = K[3];
  int32_t m = 0;
  for (int32_t v = stride / 2; v < h; v += stride)
    for (int32_t u = stride / 2; u < w; u += stride) {
      const float zf = depth[(size_t)v * w + u];
      const bool ok = std::isfinite(zf) && zf > 0.0f;
      const double z = ok ? (double)zf : 0.0;
      pts[4 * m + 0] = (u - cx) * z / fx;
      pts[4 * m + 1] = (v - cy) * z / fy;
      pts[4 * m + 2] = z;
      pts[4 * m + 3] = ok ? 1.0 : 0.0;
      ++m;
    }
  return m;
}

// ------------------------------------------------------------------------------------------------
// O4.  Trilinear TSDF sample psi(x^G)  ("query the TSDF"; A8 trilinear).
// Voxel (i,j,k) has its sample at origin + (i+1/2, j+1/2, k+1/2)*vs.  Valid iff the 2x2x2 cell is
// inside the grid and all 8 corners are observed (W > 0).  Returns 1 if valid and writes psi.
// ------------------------------------------------------------------------------------------------
static inline bool cell_ok(const orc_grid* g, const float* weight, long i, long j, long k) {
  const long X = g->dims[0], Y = g->dims[1], Z = g->dims[2];
  if (i < 0 || j < 0 || k < 0 || i + 1 > X - 1 || j + 1 > Y - 1 || k + 1 > Z - 1) return false;
  for (int c = 0; c < 8; ++c) {
    const long x = i + (c & 1), y = j + ((c >> 1) & 1), z = k + ((c >> 2) & 1);
    if (!(weight[x + X * (y + Y * z)] > 0.0f)) return false;
  }
  return true;
}

int32_t orc_trilinear(const orc_grid* g, const float* tsdf, const float* weight, const double xw[3],
                      double* psi_out, int32_t* fragile_out) {
  const long X = g->dims[0], Y = g->dims[1];
  double gc[3], f[3];
  long i0[3];
  for (int a = 0; a < 3; ++a) {
    gc[a] = (xw[a] - (double)g->origin[a]) / (double)g->voxel_size - 0.5;
    const double fl = std::floor(gc[a]);
    i0[a] = (long)fl;
    f[a] = gc[a] - fl;
  }
  const bool ok = cell_ok(g, weight, i0[0], i0[1], i0[2]);
  if (fragile_out) {
    // A26: the point is "fragile" if, within 1e-4 voxel of a cell face, the neighbouring cell has a
    // different validity (grid boundary or observed/unobserved frontier): an fp32 evaluation of the
    // same point may legitimately land on the other side.
    const double tol = 1e-4;
    int lo[3], hi[3];
    for (int a = 0; a < 3; ++a) { lo[a] = f[a] < tol ? -1 : 0; hi[a] = f[a] > 1.0 - tol ? 1 : 0; }
    bool frag = false;
    for (int dz = lo[2]; dz <= hi[2]; ++dz)
      for (int dy = lo[1]; dy <= hi[1]; ++dy)
        for (int dx = lo[0]; dx <= hi[0]; ++dx)
          if (cell_ok(g, weight, i0[0] + dx, i0[1] + dy, i0[2] + dz) != ok) frag = true;
    *fragile_out = frag ? 1 : 0;
  }
  if (!ok) return 0;
  double psi = 0;
  for (int c = 0; c < 8; ++c) {
    const int cx = c & 1, cy = (c >> 1) & 1, cz = (c >> 2) & 1;
    const double wgt = (cx ? f[0] : 1 - f[0]) * (cy ? f[1] : 1 - f[1]) * (cz ? f[2] : 1 - f[2]);
    psi += wgt * (double)tsdf[(i0[0] + cx) + X * ((i0[1] + cy) + Y * (i0[2] + cz))];
  }
  *psi_out = psi;
  return 1;
}

// ------------------------------------------------------------------------------------------------
// O5.  Fitness of one candidate pose T: S = sum over kept points of psi(R x + t)^2 (Eq. 4),
// n = number of sampled points, rho by Eq. (20) under reading A6:
//   mode 0 (F2, gated):  rho = exp(-(S + (M_O - n)) / (tau * M_O))   -- an unsampleable point of O
//                        contributes the truncation value psi^2 = 1, divisor stays |O|.
//   mode 1 (F1, option): rho = exp(-S / (tau * n)), and 0 when n < M_O/2.
// M_O = 0 -> rho = 0 (A22).
// ------------------------------------------------------------------------------------------------
double orc_rho(double S, int32_t n, int32_t M_O, int32_t mode) {
  if (M_O <= 0) return 0.0;
  if (mode == 1) {
    if (n <= 0 || 2 * (int64_t)n < (int64_t)M_O) return 0.0;
    return std::exp(-S / (ORC_TAU * (double)n));
  }
  if (mode == 2)   // "No Normalize" ablation: Eq. (14) instead of Eq. (20) -- the sum is not divided by |O|
    return std::exp(-(S + (double)(M_O - n)) / ORC_TAU);
  return std::exp(-(S + (double)(M_O - n)) / (ORC_TAU * (double)M_O));
}

static void eval_pose(const orc_grid* g, const float* tsdf, const float* weight, const double* pts,
                      const uint8_t* keep, int32_t M, const double T[12], double* S_out, int32_t* n_out,
                      int32_t* frag_out) {
  double S = 0;
  int32_t n = 0, fr = 0;
  for (int32_t i = 0; i < M; ++i) {
    if (!keep[i]) continue;
    const double* x = pts + 4 * (size_t)i;
    double xw[3];
    for (int a = 0; a < 3; ++a)                      // Eq. (1):  x^G = R x + t
      xw[a] = T[4 * a + 0] * x[0] + T[4 * a + 1] * x[1] + T[4 * a + 2] * x[2] + T[4 * a + 3];
    double psi;
    int32_t frag = 0;
    if (orc_trilinear(g, tsdf, weight, xw, &psi, &frag)) { S += psi * psi; ++n; }
    fr += frag;
  }
  *S_out = S; *n_out = n; *frag_out = fr;
}

// Candidates: if include_centre, index 0 is the centre (delta = 0) and index 1+j is particle j;
// otherwise index j is particle j.  pts: [M,4] doubles (x,y,z,mask); keep = mask != 0.
static void eval_candidates(const orc_grid* g, const float* tsdf, const float* weight, const double* pts,
                            const uint8_t* keep, int32_t M, const float* pst, int32_t N, const double T_c[12],
                            const double r[6], int include_centre, double* S, int32_t* n, int32_t* frag,
                            int nthreads) {
  const int32_t total = N + (include_centre ? 1 : 0);
  auto work = [&](int32_t lo, int32_t hi) {
    for (int32_t c = lo; c < hi; ++c) {
      double T[12];
      if (include_centre && c == 0) std::memcpy(T, T_c, sizeof(T));
      else orc_pose_from_particle(T_c, r, pst + 6 * (size_t)(c - (include_centre ? 1 : 0)), T);
      eval_pose(g, tsdf, weight, pts, keep, M, T, &S[c], &n[c], &frag[c]);
    }
  };
  if (nthreads <= 1) { work(0, total); return; }
  std::vector<std::thread> th;
  const int32_t chunk = (total + nthreads - 1) / nthreads;
  for (int t = 0; t < nthreads; ++t) {
    const int32_t lo = t * chunk, hi = std::min(total, lo + chunk);
    if (lo < hi) th.emplace_back(work, lo, hi);
  }
  for (auto& t : th) t.join();
}

// Public: rf_eval_particles equivalent (steps a2 + a3).  points float32 [M,4].
void orc_eval_particles(const orc_grid* g, const float* tsdf, const float* weight, const float* points,
                        int32_t M, const float* pst, int32_t N, const float pose[12], const float scale[6],
                        int32_t mode, int32_t nthreads, double* S_out, int32_t* n_out, int32_t* fragile_out,
                        double* rho_out, int32_t* M_O_out) {
  std::vector<double> pts(4 * (size_t)M);
  std::vector<uint8_t> keep(M);
  int32_t M_O = 0;
  for (int32_t i = 0; i < M; ++i) {
    for (int a = 0; a < 4; ++a) pts[4 * (size_t)i + a] = (double)points[4 * (size_t)i + a];
    keep[i] = points[4 * (size_t)i + 3] != 0.0f;
    M_O += keep[i];
  }
  double T_c[12], r[6];
  for (int a = 0; a < 12; ++a) T_c[a] = pose[a];
  for (int a = 0; a < 6; ++a) r[a] = scale[a];
  eval_candidates(g, tsdf, weight, pts.data(), keep.data(), M, pst, N, T_c, r, 0, S_out, n_out, fragile_out,
                  nthreads);
  for (int32_t j = 0; j < N; ++j) rho_out[j] = orc_rho(S_out[j], n_out[j], M_O, mode);
  *M_O_out = M_O;
}

// ------------------------------------------------------------------------------------------------
// O6.  Overlap pixel set O_k (Eq. 19; recomputed every iteration with s*_{k-1}):
// point i is kept iff, moved to the world by T_km1 and into camera t-1 (pose T_prev), it has z > 0
// and projects inside [0,W) x [0,H)   (A9: rectangle + positive z only).
// ------------------------------------------------------------------------------------------------
int32_t orc_overlap_mask(const double* pts, int32_t M, const double T_km1[12], const double T_prev[12],
                         const float K[4], int32_t w, int32_t h, uint8_t* keep) {
  const double fx = K[0], fy = K[1], cx = K[2], cy = K[3];
  int32_t cnt = 0;
  for (int32_t i = 0; i < M; ++i) {
    const double* x = pts + 4 * (size_t)i;
    keep[i] = 0;
    if (x[3] == 0.0) continue;
    double xw[3], y[3];
    for (int a = 0; a < 3; ++a)
      xw[a] = T_km1[4 * a + 0] * x[0] + T_km1[4 * a + 1] * x[1] + T_km1[4 * a + 2] * x[2] + T_km1[4 * a + 3];
    for (int a = 0; a < 3; ++a)   // y = R_prev^T (x^G - t_prev)
      y[a] = T_prev[0 + a] * (xw[0] - T_prev[3]) + T_prev[4 + a] * (xw[1] - T_prev[7]) +
             T_prev[8 + a] * (xw[2] - T_prev[11]);
    if (!(y[2] > 0.0)) continue;
    const double u = fx * y[0] / y[2] + cx, v = fy * y[1] / y[2] + cy;
    if (u >= 0.0 && u < (double)w && v >= 0.0 && v < (double)h) { keep[i] = 1; ++cnt; }
  }
  return cnt;
}

// ------------------------------------------------------------------------------------------------
// O7 steps 3-6.  Swarm update from the fitness values of one iteration (P:L229-260, P:L292,
// P:L300-304).  rho[0] is the centre s*_{k-1} (A14), rho[1+j] particle j.
// Outputs: T_new, r_new, trace fields.  Returns the stop code: 0 continue, 1 two empty APS in a
// row, 2 change < 1e-6 in all six dims (non-empty APS only, A16).  (The k = K cap is the caller's.)
// ------------------------------------------------------------------------------------------------
struct orc_update_out {
  double T_new[12];
  double r_new[6];
  double delta_star[6];
  double rho_ref, rho_max, rho_tilde, sum_omega;
  int32_t n_aps, argmax, empty_run, stop;
};

// Ablation variants of SURVEY 8(f)-1 (Fig. 11; Table 2).  Bits of `variant`:
//   ORC_VAR_NO_OVERLAP     O_k := every valid pixel of I_d ("No Overlap": "replacing O^t by I_d^t in Eq. (20)")
//   ORC_VAR_RESCALE_ISO    Eq. (17) with its isotropic part only:   r^_d = (1 - rho~) / sqrt(6) + eps
//   ORC_VAR_RESCALE_ANISO  Eq. (17) with its anisotropic part only: r^_d = |v_d| / ||v|| + eps
// ("anisotropic part ... the attractor v, and an isotropic part ... 1 - rho(s_k^*)").  The empty-APS rule
// has no direction and is left as it is in every variant.
//   ORC_VAR_THRESH_EQ21    A14 variant: the advantage-set threshold rho(s*_{k-1}) is not re-evaluated but taken
//                          from the previous iteration -- Eq. (21)'s estimate rho~ of the step that produced s*_{k-1}
//                          (or, after an empty step, the threshold that step used).  The first iteration of a frame has
//                          no previous one and evaluates the centre exactly.  `thresh` carries it; NaN = evaluate (rho[0]).
static const int32_t ORC_VAR_NO_OVERLAP = 1, ORC_VAR_RESCALE_ISO = 2, ORC_VAR_RESCALE_ANISO = 4, ORC_VAR_THRESH_EQ21 = 8;

void orc_swarm_update_t(const double* rho, const float* pst, int32_t N, const double T[12], const double r[6],
                        int32_t empty_run_in, int32_t variant, double thresh, orc_update_out* o) {
  const double rho_ref = ((variant & ORC_VAR_THRESH_EQ21) && !std::isnan(thresh)) ? thresh : rho[0];
  int32_t best = 0;
  for (int32_t c = 1; c <= N; ++c) if (rho[c] > rho[best]) best = c;      // ties -> lowest index (A18)
  // Advantage Particle Set: strictly better than s*_{k-1}.
  double sum_w = 0;
  int32_t n_aps = 0;
  for (int32_t j = 0; j < N; ++j) if (rho[1 + j] > rho_ref) { sum_w += rho[1 + j] - rho_ref; ++n_aps; }
  double dstar[6] = {0, 0, 0, 0, 0, 0}, rho_tilde = 0, rhat[6];
  if (n_aps > 0) {
    for (int32_t j = 0; j < N; ++j) {
      if (!(rho[1 + j] > rho_ref)) continue;
      const double wbar = (rho[1 + j] - rho_ref) / sum_w;                    // Eq. (15) weights
      for (int d = 0; d < 6; ++d) dstar[d] += wbar * (r[d] * (double)pst[6 * (size_t)j + d]);   // Eq. (15), A3
      rho_tilde += wbar * rho[1 + j];                                        // Eq. (21)
    }
    orc_apply_delta(T, dstar, o->T_new);                                     // MovePST
    double nv = 0;
    for (int d = 0; d < 6; ++d) nv += dstar[d] * dstar[d];                   // v = s_k^* - s_{k-1}^*  (Eq. 16)
    nv = std::sqrt(nv);
    for (int d = 0; d < 6; ++d) {                                            // Eq. (17), A4 (abs), A5
      const double aniso = nv > 0 ? std::fabs(dstar[d]) / nv : 0.0, iso = 1.0 - rho_tilde;
      if (variant & ORC_VAR_RESCALE_ISO) rhat[d] = iso / std::sqrt(6.0) + ORC_EPS;
      else if (variant & ORC_VAR_RESCALE_ANISO) rhat[d] = aniso + ORC_EPS;
      else rhat[d] = (nv > 0 ? (1.0 - rho_tilde) * std::fabs(dstar[d]) / nv : 0.0) + ORC_EPS;
    }
    o->empty_run = 0;
  } else {
    std::memcpy(o->T_new, T, sizeof(double) * 12);
    for (int d = 0; d < 6; ++d) rhat[d] = 2.0 * (1.0 - rho_ref) / std::sqrt(6.0) + ORC_EPS;   // P:L292, A13
    o->empty_run = empty_run_in + 1;
  }
  for (int d = 0; d < 6; ++d) o->r_new[d] = ORC_BETA * r[d] + (1.0 - ORC_BETA) * rhat[d];      // Eq. (18)
  std::memcpy(o->delta_star, dstar, sizeof(dstar));
  o->rho_ref = rho_ref; o->rho_max = rho[best]; o->rho_tilde = rho_tilde; o->sum_omega = sum_w;
  o->n_aps = n_aps; o->argmax = best;
  o->stop = 0;
  if (o->empty_run >= ORC_EMPTY_STOP) o->stop = 1;
  else if (n_aps > 0) {
    double mx = 0;
    for (int d = 0; d < 6; ++d) mx = std::max(mx, std::fabs(dstar[d]));
    if (mx < ORC_STOP) o->stop = 2;
  }
}

void orc_swarm_update_v(const double* rho, const float* pst, int32_t N, const double T[12], const double r[6],
                        int32_t empty_run_in, int32_t variant, orc_update_out* o) {
  orc_swarm_update_t(rho, pst, N, T, r, empty_run_in, variant, std::numeric_limits<double>::quiet_NaN(), o);
}

void orc_swarm_update(const double* rho, const float* pst, int32_t N, const double T[12], const double r[6],
                      int32_t empty_run_in, orc_update_out* o) {
  orc_swarm_update_v(rho, pst, N, T, r, empty_run_in, 0, o);
}

// Every valid point, whatever the poses ("No Overlap" ablation).
static int32_t all_valid_mask(const double* pts, int32_t M, uint8_t* keep) {
  int32_t cnt = 0;
  for (int32_t i = 0; i < M; ++i) { keep[i] = pts[4 * (size_t)i + 3] != 0.0; cnt += keep[i]; }
  return cnt;
}

// ------------------------------------------------------------------------------------------------
// O7 + O8 (tracking part).  Algorithm 1 for one frame against a fixed volume.
// Levels l = (k-1) mod 3 in the listed order (A15): (pst[0], stride[0]), (pst[1], stride[1]), ...
// Trace arrays have `iters` rows.  early_stop = 0 forces exactly `iters` iterations (config 2).
// Returns the number of iterations run.
// ------------------------------------------------------------------------------------------------
struct orc_trace_row {
  int32_t level, M_O, n_aps, argmax, stop, empty_run;
  double rho_ref, rho_max, rho_tilde, sum_omega;
  double delta_star[6];
  double pose[12];
  double r[6];
};

int32_t orc_pfo_track_v(const orc_grid* g, const float* tsdf, const float* weight, const float* depth, int32_t w,
                        int32_t h, const float K[4], const float* const pst[3], const int32_t N[3],
                        const int32_t stride[3], int32_t iters, int32_t early_stop, int32_t mode, int32_t variant,
                        int32_t nthreads, double pose_io[12], const double prev_pose[12], double r0_io[6],
                        int32_t* has_r0_io, orc_trace_row* trace /* [iters] or NULL */, double* final_rho,
                        int32_t* final_count, int64_t* evals_out) {
  // a0: back-project the three levels once.
  std::vector<double> pts[3];
  int32_t M[3];
  for (int l = 0; l < 3; ++l) {
    pts[l].resize(4 * (size_t)orc_lattice_count(w, stride[l]) * orc_lattice_count(h, stride[l]) + 4);
    M[l] = orc_backproject(depth, w, h, K, stride[l], pts[l].data());
  }
  double T[12], r[6];
  std::memcpy(T, pose_io, sizeof(T));
  int64_t evals = 0;
  std::vector<uint8_t> keep;
  std::vector<double> S, rho;
  std::vector<int32_t> n, frag;
  if (!*has_r0_io) {
    // A11: first tracked frame -- evaluate the centre alone on level 0, isotropic r0 from P:L292.
    keep.assign(M[0], 0);
    const int32_t M_O = (variant & ORC_VAR_NO_OVERLAP) ? all_valid_mask(pts[0].data(), M[0], keep.data())
                                                       : orc_overlap_mask(pts[0].data(), M[0], T, prev_pose, K, w, h, keep.data());
    double S0; int32_t n0, f0;
    eval_pose(g, tsdf, weight, pts[0].data(), keep.data(), M[0], T, &S0, &n0, &f0);
    const double rho0 = orc_rho(S0, n0, M_O, mode);
    for (int d = 0; d < 6; ++d) r[d] = 2.0 * (1.0 - rho0) / std::sqrt(6.0) + ORC_EPS;
    evals += M_O;
  } else {
    std::memcpy(r, r0_io, sizeof(r));
  }
  int32_t empty_run = 0, k_run = 0;
  double last_rho = 0; int32_t last_cnt = 0;
  double thresh = std::numeric_limits<double>::quiet_NaN();          // A14 variant: threshold carried between iterations
  for (int32_t k = 1; k <= iters; ++k) {
    const int l = (k - 1) % 3;
    keep.assign(M[l], 0);
    const int32_t M_O = (variant & ORC_VAR_NO_OVERLAP) ? all_valid_mask(pts[l].data(), M[l], keep.data())
                                                       : orc_overlap_mask(pts[l].data(), M[l], T, prev_pose, K, w, h, keep.data());   // O6
    S.assign(N[l] + 1, 0); n.assign(N[l] + 1, 0); frag.assign(N[l] + 1, 0); rho.assign(N[l] + 1, 0);
    eval_candidates(g, tsdf, weight, pts[l].data(), keep.data(), M[l], pst[l], N[l], T, r, 1, S.data(), n.data(),
                    frag.data(), nthreads);
    for (int32_t c = 0; c <= N[l]; ++c) rho[c] = orc_rho(S[c], n[c], M_O, mode);
    evals += (int64_t)(N[l] + 1) * M_O;
    orc_update_out u;
    orc_swarm_update_t(rho.data(), pst[l], N[l], T, r, empty_run, variant, thresh, &u);
    if (variant & ORC_VAR_THRESH_EQ21) thresh = u.n_aps > 0 ? u.rho_tilde : u.rho_ref;
    std::memcpy(T, u.T_new, sizeof(T));
    std::memcpy(r, u.r_new, sizeof(r));
    empty_run = u.empty_run;
    if (k == 1) { std::memcpy(r0_io, r, sizeof(r)); *has_r0_io = 1; }       // P:L286  r_0^{t+1} = r_1^t
    last_rho = u.n_aps > 0 ? u.rho_tilde : u.rho_ref;
    last_cnt = n[u.argmax];
    k_run = k;
    if (trace) {
      orc_trace_row& tr = trace[k - 1];
      tr.level = l; tr.M_O = M_O; tr.n_aps = u.n_aps; tr.argmax = u.argmax; tr.stop = u.stop; tr.empty_run = u.empty_run;
      tr.rho_ref = u.rho_ref; tr.rho_max = u.rho_max; tr.rho_tilde = u.rho_tilde; tr.sum_omega = u.sum_omega;
      std::memcpy(tr.delta_star, u.delta_star, sizeof(tr.delta_star));
      std::memcpy(tr.pose, T, sizeof(T));
      std::memcpy(tr.r, r, sizeof(r));
    }
    if (early_stop && u.stop) break;
  }
  std::memcpy(pose_io, T, sizeof(T));
  if (final_rho) *final_rho = last_rho;
  if (final_count) *final_count = last_cnt;
  if (evals_out) *evals_out = evals;
  return k_run;
}

int32_t orc_pfo_track(const orc_grid* g, const float* tsdf, const float* weight, const float* depth, int32_t w,
                      int32_t h, const float K[4], const float* const pst[3], const int32_t N[3],
                      const int32_t stride[3], int32_t iters, int32_t early_stop, int32_t mode, int32_t nthreads,
                      double pose_io[12], const double prev_pose[12], double r0_io[6], int32_t* has_r0_io,
                      orc_trace_row* trace /* [iters] or NULL */, double* final_rho, int32_t* final_count,
                      int64_t* evals_out) {
  return orc_pfo_track_v(g, tsdf, weight, depth, w, h, K, pst, N, stride, iters, early_stop, mode, 0, nthreads, pose_io,
                         prev_pose, r0_io, has_r0_io, trace, final_rho, final_count, evals_out);
}

// ------------------------------------------------------------------------------------------------
// Baselines of the paper's comparison in Section 5.2 (Fig. 9, 10): "vanilla PFO" (Section 3.2)
// and particle swarm optimisation, on the same fitness (Eq. 20 under reading A6) and the same pose chart as
// Algorithm 1: a particle is a 6-D increment delta (imaginary quaternion part, translation) about the frame's initial
// pose T_0, candidate pose = Delta(delta) o T_0 (A2, A3).  Every random number the methods draw is an INPUT, so that
// the oracle and the CUDA path consume the same stream.
// Readings (the paper gives no constants for its baselines): B1 systematic resampling; B2 the PSO
// constants of Clerc & Kennedy; B3 increments are clamped to |delta_q| <= 0.95 so that they stay rigid motions; B4 the
// particle state is stored in binary32 (the paper keeps particles in GPU memory): every update below is
// evaluated in fp64 from binary32 operands, in the written order, and rounded once; B5 the overlap set is the one of the
// frame's initial pose s^{t-1}, i.e. every valid pixel (Eq. 19 with both poses equal).  Parity with the authors' baselines
// is unpinned.
// ------------------------------------------------------------------------------------------------
// Fitness of N explicit increments (binary32) about T_0 on a point set; keep = every valid point (B5).
static void eval_increments(const orc_grid* g, const float* tsdf, const float* weight, const double* pts, int32_t M,
                            const uint8_t* keep, int32_t M_O, const float* delta /*[N,6]*/, int32_t N,
                            const double T0[12], int32_t mode, int32_t nthreads, double* rho) {
  auto work = [&](int32_t lo, int32_t hi) {
    for (int32_t i = lo; i < hi; ++i) {
      double T[12], S, d[6]; int32_t n, fr;
      for (int a = 0; a < 6; ++a) d[a] = (double)delta[6 * (size_t)i + a];
      orc_apply_delta(T0, d, T);
      eval_pose(g, tsdf, weight, pts, keep, M, T, &S, &n, &fr);
      rho[i] = orc_rho(S, n, M_O, mode);
    }
  };
  if (nthreads <= 1) { work(0, N); return; }
  std::vector<std::thread> th;
  const int32_t chunk = (N + nthreads - 1) / nthreads;
  for (int t = 0; t < nthreads; ++t) {
    const int32_t lo = t * chunk, hi = std::min(N, lo + chunk);
    if (lo < hi) th.emplace_back(work, lo, hi);
  }
  for (auto& t : th) t.join();
}

// B3: keep an increment a valid rigid motion -- |delta_q| <= 0.95 (radial clamp of the quaternion block), then B4.
static inline void clamp_and_store(double d[6], float* out) {
  const double q_max = 0.95;
  const double n = std::sqrt((d[0] * d[0] + d[1] * d[1]) + d[2] * d[2]);
  if (n > q_max) { const double sc = q_max / n; for (int a = 0; a < 3; ++a) d[a] = d[a] * sc; }
  for (int a = 0; a < 6; ++a) out[a] = (float)d[a];
}

// Eq. (12): delta_out_i = clamp(delta_in_{a(i)} + sigma (.) z_i), a = ancestors (NULL: identity).
void orc_baseline_propose(const float* delta_in, const int32_t* ancestors, const float sigma[6], const float* normals,
                          int32_t N, float* delta_out) {
  for (int32_t i = 0; i < N; ++i) {
    const int32_t a0 = ancestors ? ancestors[i] : i;
    double d[6];
    for (int a = 0; a < 6; ++a) d[a] = (double)delta_in[6 * (size_t)a0 + a] + (double)sigma[a] * (double)normals[6 * (size_t)i + a];
    clamp_and_store(d, delta_out + 6 * (size_t)i);
  }
}

// Systematic resampling (B1): N slots at u_m = (m + u) / N, ancestor of slot m = first i with C_i > u_m, where C is the
// running sum of the normalised weights w_i / sum(w) (fp64, index order; Eq. 13: the weight of a particle is its
// likelihood, the prior weights being uniform after the previous resampling).  near_out (optional): 1 for slots whose u_m
// lies within `tol` of a boundary C_i -- a path whose weights differ within the fitness tolerance may pick the neighbour.
void orc_systematic_resample(const double* w, int32_t N, double u, double tol, int32_t* ancestor, uint8_t* near_out) {
  double tot = 0;
  for (int32_t i = 0; i < N; ++i) tot += w[i];
  std::vector<double> C(N);
  double run = 0;
  for (int32_t i = 0; i < N; ++i) { run += w[i] / tot; C[i] = run; }
  C[N - 1] = 2.0;                                          // the last particle closes the unit interval whatever the rounding
  int32_t i = 0;
  for (int32_t m = 0; m < N; ++m) {
    const double um = ((double)m + u) / (double)N;
    while (C[i] <= um) ++i;
    ancestor[m] = i;
    if (near_out) {
      const double lo = i > 0 ? C[i - 1] : 0.0;
      near_out[m] = (um - lo < tol || (i < N - 1 && C[i] - um < tol)) ? 1 : 0;
    }
  }
}

// PSO with inertia weight (the constriction constants of Clerc & Kennedy 2002, B2): omega = 0.7298, c1 = c2 = 1.49618.
//   v_i <- omega v_i + c1 a_i (.) (p_i - x_i) + c2 b_i (.) (gbest - x_i);   x_i <- clamp(x_i + v_i)   (B3, B4)
// with a, b uniform in [0,1)^6 (inputs), p_i the particle's best position so far, gbest the swarm's.
static const double ORC_PSO_OMEGA = 0.7298, ORC_PSO_C = 1.49618;
double orc_pso_const(int which) { return which == 0 ? ORC_PSO_OMEGA : ORC_PSO_C; }

void orc_baseline_pso_move(float* x, float* v, const float* pbest, const float gbest[6], const float* ua, const float* ub, int32_t N) {
  for (int32_t i = 0; i < N; ++i) {
    double d[6];
    for (int a = 0; a < 6; ++a) {
      const size_t q = 6 * (size_t)i + a;
      const double xi = (double)x[q];
      const double t1 = ORC_PSO_OMEGA * (double)v[q];
      const double t2 = (ORC_PSO_C * (double)ua[q]) * ((double)pbest[q] - xi);
      const double t3 = (ORC_PSO_C * (double)ub[q]) * ((double)gbest[a] - xi);
      v[q] = (float)((t1 + t2) + t3);
      d[a] = xi + (double)v[q];
    }
    clamp_and_store(d, x + 6 * (size_t)i);
  }
}

// Best-so-far bookkeeping shared by the two baselines: personal bests (optional) and the swarm / run best, strict > so
// that ties keep the earlier holder; among the particles of one step the lowest index wins (A18).
// gbest: [8] = 6 coordinates, fitness, index (as a float).  first != 0: initialise from this step.
void orc_baseline_best(const float* fitness, const float* x, int32_t N, float* pbest, float* pbest_fit, int32_t first, float gbest[8]) {
  int32_t bi = 0;
  for (int32_t i = 0; i < N; ++i) {
    if (pbest && (first || fitness[i] > pbest_fit[i])) { pbest_fit[i] = fitness[i]; std::memcpy(pbest + 6 * (size_t)i, x + 6 * (size_t)i, 6 * sizeof(float)); }
    if (fitness[i] > fitness[bi]) bi = i;
  }
  if (first || fitness[bi] > gbest[6]) { std::memcpy(gbest, x + 6 * (size_t)bi, 6 * sizeof(float)); gbest[6] = fitness[bi]; gbest[7] = (float)bi; }
}

// Fitness of explicit increments, the oracle counterpart of rf_eval_particles with scale = 1 (B5: every valid point).
void orc_eval_increments(const orc_grid* g, const float* tsdf, const float* weight, const float* points, int32_t M,
                         const float* delta, int32_t N, const float pose[12], int32_t mode, int32_t nthreads, double* rho_out) {
  std::vector<double> pts(4 * (size_t)M);
  std::vector<uint8_t> keep(M);
  int32_t M_O = 0;
  for (int32_t i = 0; i < M; ++i) {
    for (int a = 0; a < 4; ++a) pts[4 * (size_t)i + a] = (double)points[4 * (size_t)i + a];
    keep[i] = points[4 * (size_t)i + 3] != 0.0f;
    M_O += keep[i];
  }
  double T0[12];
  for (int a = 0; a < 12; ++a) T0[a] = pose[a];
  eval_increments(g, tsdf, weight, pts.data(), M, keep.data(), M_O, delta, N, T0, mode, nthreads, rho_out);
}

// ------------------------------------------------------------------------------------------------
// O9.  Projective TSDF integration (volumetric depth fusion framework [Curless-Levoy 1996; Izadi
// 2011] cited at P:L81; 3 ms/frame P:L545; the paper gives no formula -> reading A17).
// The definition, written out in fp64, per voxel (i,j,k):
//   p_w = origin + (i+1/2, j+1/2, k+1/2) * vs                  voxel centre (world)
//   p_c = R^T (p_w - t)                                         into the camera frame (inverse of Eq. 1)
//   skip if p_c.z <= 0
//   u = floor(fx * p_c.x / p_c.z + cx + 1/2),  v likewise       nearest pixel (pixel centres at integers)
//   skip if (u,v) outside [0,W) x [0,H);  d = D[v,u];  skip if d <= 0 or non-finite
//   sdf = d - p_c.z;  skip if sdf < -mu
//   f = min(1, sdf / mu);  F <- (W F + f) / (W + 1);  W <- min(W + 1, W_max)
// half_storage != 0: F is rounded to binary16 (round-to-nearest-even) after every update.
//
// Fragile voxels (the integration counterpart of A26; DESIGN.md section 3 reading R-I2, which retires R-I1):
// three decisions above turn a real number into an integer or a branch (z > 0, the pixel (u,v), sdf >= -mu).  A binary32
// evaluation of p_c is within eps_p = 2e-6 m of the fp64 one in each component (binary32 spacing at 8-16 m is 9.5e-7;
// two roundings at that magnitude), so it may take the other side of a decision that lies within that reach.  The
// oracle flags a voxel (fragile_out, 0/1 per voxel, optional) when
//   |p_c.z| <= eps_p,  or
//   the pixel changes when the projection moves by eps_p * f * (1 + |x/z|) / z  (resp. y, fy) in either direction and
//   one of the two candidate pixels lies inside the image,  or
//   the voxel reaches the band test and |sdf + mu| <= eps_p + 2^-22 * d   (the depth value itself is binary32).
// Parity gate: weights exact and values within tolerance on every voxel that is not flagged; flagged voxels are
// counted (expected < 1 %) and only checked for being one update apart at most.
// ------------------------------------------------------------------------------------------------
static float round_to_half(double v) {
  // software binary16 rounding (round-to-nearest-even) of a finite value of magnitude <= 1:
  // quantum 2^(e-10) for normal halves (e >= -14), 2^-24 in the subnormal range.
  if (v == 0.0 || !std::isfinite(v)) return (float)v;
  int e;
  std::frexp(std::fabs(v), &e);
  e -= 1;                                   // |v| = m * 2^e with m in [1,2)
  if (e < -14) e = -14;
  const double q = std::ldexp(1.0, e - 10);
  return (float)std::copysign(std::nearbyint(std::fabs(v) / q) * q, v);   // default mode = RNE
}

float orc_round_to_half(double v) { return round_to_half(v); }

static const double ORC_EPS_P = 2e-6;    // metres; reach of a binary32 evaluation of p_c (see above)

double orc_integrate_eps_p(void) { return ORC_EPS_P; }

static inline void integ_voxel(const orc_grid* g, const float K[4], const float pose[12], const float* depth,
                               int32_t w, int32_t h, int i, int j, int k, float w_max, int half_storage, float* F,
                               float* W, uint8_t* fragile) {
  const double vs = g->voxel_size, mu = g->trunc;
  const double fx = K[0], fy = K[1], cx = K[2], cy = K[3];
  const double idx[3] = {(double)i, (double)j, (double)k};
  double pw[3], pc[3];
  for (int a = 0; a < 3; ++a) pw[a] = (double)g->origin[a] + (idx[a] + 0.5) * vs;
  for (int a = 0; a < 3; ++a) {              // p_c = R^T (p_w - t): component a uses column a of R
    pc[a] = 0;
    for (int b = 0; b < 3; ++b) pc[a] += (double)pose[4 * b + a] * (pw[b] - (double)pose[4 * b + 3]);
  }
  const double z = pc[2];
  if (fragile && std::fabs(z) <= ORC_EPS_P) *fragile = 1;
  if (!(z > 0.0)) return;
  const double uf = fx * pc[0] / z + cx, vf = fy * pc[1] / z + cy;
  const double ur = std::floor(uf + 0.5), vr = std::floor(vf + 0.5);
  if (fragile) {
    const double du = ORC_EPS_P * fx * (1.0 + std::fabs(pc[0] / z)) / z, dv = ORC_EPS_P * fy * (1.0 + std::fabs(pc[1] / z)) / z;
    const double u0 = std::floor(uf + 0.5 - du), u1 = std::floor(uf + 0.5 + du);
    const double v0 = std::floor(vf + 0.5 - dv), v1 = std::floor(vf + 0.5 + dv);
    const bool hits = u1 >= 0.0 && u0 < (double)w && v1 >= 0.0 && v0 < (double)h;   // some candidate pixel is in the image
    if ((u0 != u1 || v0 != v1) && hits) *fragile = 1;
  }
  if (!(ur >= 0.0 && ur < (double)w && vr >= 0.0 && vr < (double)h)) return;
  const float df = depth[(size_t)(long)vr * w + (long)ur];
  if (!(std::isfinite(df) && df > 0.0f)) return;
  const double d = (double)df;
  const double sdf = d - z;
  if (fragile && std::fabs(sdf + mu) <= ORC_EPS_P + std::ldexp(d, -22)) *fragile = 1;
  if (sdf < -mu) return;
  const double f = std::min(1.0, sdf / mu);
  const double Wd = *W;
  const double Fold = Wd > 0 ? (double)*F : 0.0;
  const double Fn = (Wd * Fold + f) / (Wd + 1.0);
  *F = half_storage ? round_to_half(Fn) : (float)Fn;
  *W = std::min(*W + 1.0f, w_max);
}

// fragile_out: NULL, or X*Y*Z bytes that are SET to 1 for voxels flagged in this frame (never cleared here, so a
// caller can accumulate over frames).
void orc_integrate(const orc_grid* g, float* tsdf, float* weight, const float* depth, int32_t w, int32_t h,
                   const float K[4], const float pose[12], int32_t w_max, int32_t half_storage, int32_t nthreads,
                   uint8_t* fragile_out) {
  const int X = g->dims[0], Y = g->dims[1], Z = g->dims[2];
  auto work = [&](int z0, int z1) {
    for (int k = z0; k < z1; ++k)
      for (int j = 0; j < Y; ++j)
        for (int i = 0; i < X; ++i) {
          const size_t idx = (size_t)i + (size_t)X * ((size_t)j + (size_t)Y * k);
          integ_voxel(g, K, pose, depth, w, h, i, j, k, (float)w_max, half_storage, &tsdf[idx], &weight[idx],
                      fragile_out ? &fragile_out[idx] : nullptr);
        }
  };
  if (nthreads <= 1) { work(0, Z); return; }
  std::vector<std::thread> th;
  const int chunk = (Z + nthreads - 1) / nthreads;
  for (int t = 0; t < nthreads; ++t) {
    const int z0 = t * chunk, z1 = std::min(Z, z0 + chunk);
    if (z0 < z1) th.emplace_back(work, z0, z1);
  }
  for (auto& t : th) t.join();
}

// Same update restricted to a list of voxels (voxels are independent): lin[i] = x + X*(y + Y*z);
// tsdf_sub / weight_sub / fragile_sub hold the state of exactly those voxels.  Used for config 5 (1024^3).
void orc_integrate_subset(const orc_grid* g, const int64_t* lin, int64_t count, float* tsdf_sub, float* weight_sub,
                          const float* depth, int32_t w, int32_t h, const float K[4], const float pose[12],
                          int32_t w_max, int32_t half_storage, uint8_t* fragile_sub) {
  const int64_t X = g->dims[0], Y = g->dims[1];
  for (int64_t q = 0; q < count; ++q) {
    const int i = (int)(lin[q] % X), j = (int)((lin[q] / X) % Y), k = (int)(lin[q] / (X * Y));
    integ_voxel(g, K, pose, depth, w, h, i, j, k, (float)w_max, half_storage, &tsdf_sub[q], &weight_sub[q],
                fragile_sub ? &fragile_sub[q] : nullptr);
  }
}

// ------------------------------------------------------------------------------------------------
// O9.  Read-out of the fused surface by ray casting (the paper shows reconstructions,
// P:L525-537, and gives no read-out algorithm: reading R-R1 in DESIGN.md).
// Pixel (u,v) looks along x_c(z) = ((u-cx)/fx, (v-cy)/fy, 1) * z  (P:L93 back-projection, depth-parametrised), world
// point x(z) = R x_c(z) + t (Eq. 1).  Samples psi_k = psi(x(k*step)), k = 1 .. floor(z_max/step), in order; the surface
// is the first k at which samples k-1 and k are both valid (O4) with psi_{k-1} > 0 >= psi_k; its depth is the zero of
// the straight line through the two samples, z* = (k-1)*step + step * psi_{k-1} / (psi_{k-1} - psi_k).
// No such k -> depth 0.  A crossing from behind (negative to positive) is not a surface.
// Normal (optional): gradient of psi at x(z*) by central differences of half-width one voxel along the world axes,
// normalised; NaN if any of the six samples is invalid or the gradient is zero.
// fragile_out (optional, per pixel): 1 if any sample up to the hit was fragile in the sense of A26, or the crossing's
// denominator psi_{k-1} - psi_k is below 1e-3, or a sample of the march lies within 1e-5 of zero (the fp32 kernel
// may take the neighbouring interval): such pixels are excluded from the tight comparison and counted.
// ------------------------------------------------------------------------------------------------
void orc_raycast(const orc_grid* g, const float* tsdf, const float* weight, const float K[4], int32_t w, int32_t h,
                 const float pose[12], double step, double z_max, double* depth_out, double* normal_out,
                 uint8_t* fragile_out, int32_t nthreads) {
  const double fx = K[0], fy = K[1], cx = K[2], cy = K[3];
  const long nk = (long)std::floor(z_max / step);
  auto world = [&](int u, int v, double z, double x[3]) {
    const double xc[3] = {(u - cx) / fx * z, (v - cy) / fy * z, z};
    for (int a = 0; a < 3; ++a)
      x[a] = (double)pose[4 * a + 0] * xc[0] + (double)pose[4 * a + 1] * xc[1] + (double)pose[4 * a + 2] * xc[2] + (double)pose[4 * a + 3];
  };
  auto rows = [&](int v0, int v1) {
    for (int v = v0; v < v1; ++v)
      for (int u = 0; u < w; ++u) {
        const size_t pix = (size_t)v * w + u;
        bool prev_ok = false, frag = false;
        double prev = 0, zhit = 0;
        for (long k = 1; k <= nk; ++k) {
          double x[3], psi = 0;
          int32_t fr = 0;
          world(u, v, (double)k * step, x);
          const bool ok = orc_trilinear(g, tsdf, weight, x, &psi, &fr) != 0;
          if (fr) frag = true;
          if (ok && std::fabs(psi) < 1e-5) frag = true;
          if (ok && prev_ok && prev > 0.0 && psi <= 0.0) {
            if (prev - psi < 1e-3) frag = true;
            zhit = (double)(k - 1) * step + step * prev / (prev - psi);
            break;
          }
          prev_ok = ok;
          prev = psi;
        }
        depth_out[pix] = zhit;
        if (normal_out) {
          double n[3] = {NAN, NAN, NAN};
          if (zhit > 0) {
            double x[3], grad[3];
            world(u, v, zhit, x);
            bool all = true;
            for (int a = 0; a < 3 && all; ++a) {
              double xp[3] = {x[0], x[1], x[2]}, xm[3] = {x[0], x[1], x[2]}, fp = 0, fm = 0;
              int32_t f1 = 0, f2 = 0;
              xp[a] += (double)g->voxel_size;
              xm[a] -= (double)g->voxel_size;
              all = orc_trilinear(g, tsdf, weight, xp, &fp, &f1) && orc_trilinear(g, tsdf, weight, xm, &fm, &f2);
              if (f1 || f2) frag = true;
              grad[a] = fp - fm;
            }
            const double len = all ? std::sqrt(grad[0] * grad[0] + grad[1] * grad[1] + grad[2] * grad[2]) : 0.0;
            if (all && len > 0) for (int a = 0; a < 3; ++a) n[a] = grad[a] / len;
          }
          for (int a = 0; a < 3; ++a) normal_out[3 * pix + a] = n[a];
        }
        if (fragile_out) fragile_out[pix] = frag ? 1 : 0;
      }
  };
  if (nthreads <= 1) { rows(0, h); return; }
  std::vector<std::thread> th;
  const int chunk = (h + nthreads - 1) / nthreads;
  for (int t = 0; t < nthreads; ++t) {
    const int v0 = t * chunk, v1 = std::min((int)h, v0 + chunk);
    if (v0 < v1) th.emplace_back(rows, v0, v1);
  }
  for (auto& t : th) t.join();
}

// ------------------------------------------------------------------------------------------------
// O10.  Surface point set of the fused TSDF ("marching cubes ... to point sets", the reconstruction whose
// completeness / accuracy the paper measures; reading R-R2 in DESIGN.md).  The vertex set of marching cubes: every
// grid edge between voxel a = (i,j,k) and its +x, +y or +z neighbour b whose two samples are both observed (W > 0) and lie
// on different sides of the surface -- exactly one of psi_a, psi_b is > 0 -- carries one point, the zero of the straight
// line through the two samples:  p = c_a + t (c_b - c_a),  t = psi_a / (psi_a - psi_b),  c = voxel centre.
// Output in scan order (k, j, i, then axis x, y, z): points [n,3] doubles and the edge key 3 * (i + X (j + Y k)) + axis.
// Returns the number of crossing edges; at most `cap` are written.
// ------------------------------------------------------------------------------------------------
int64_t orc_surface_points(const orc_grid* g, const float* tsdf, const float* weight, double* points_out, int64_t* edge_out,
                           int64_t cap) {
  const int64_t X = g->dims[0], Y = g->dims[1], Z = g->dims[2];
  const double vs = g->voxel_size;
  int64_t n = 0;
  for (int64_t k = 0; k < Z; ++k)
    for (int64_t j = 0; j < Y; ++j)
      for (int64_t i = 0; i < X; ++i) {
        const int64_t a = i + X * (j + Y * k);
        if (!(weight[a] > 0.0f)) continue;
        const double pa = tsdf[a];
        const int64_t nb[3] = {i + 1 < X ? a + 1 : -1, j + 1 < Y ? a + X : -1, k + 1 < Z ? a + X * Y : -1};
        for (int d = 0; d < 3; ++d) {
          if (nb[d] < 0 || !(weight[nb[d]] > 0.0f)) continue;
          const double pb = tsdf[nb[d]];
          if ((pa > 0.0) == (pb > 0.0)) continue;
          if (n < cap) {
            const double t = pa / (pa - pb);
            double c[3] = {(double)g->origin[0] + ((double)i + 0.5) * vs, (double)g->origin[1] + ((double)j + 0.5) * vs,
                           (double)g->origin[2] + ((double)k + 0.5) * vs};
            c[d] += t * vs;
            for (int q = 0; q < 3; ++q) points_out[3 * n + q] = c[q];
            if (edge_out) edge_out[n] = 3 * a + d;
          }
          ++n;
        }
      }
  return n;
}

// ------------------------------------------------------------------------------------------------
// O11.  Gauss-Newton minimisation of Eq. (4) (the tracker of [Bylow 2013] that the paper compares with,
// "they ... employ the Gauss-Newton method to minimize the summation of TSDF").  Same objective
// and sample rule as the fitness (O4, O5): E(T) = sum over valid points of psi(R x + t)^2.  Reading GN1:
//   residual   r_i = psi(p_i),  p_i = R x_i + t                                (points that cannot be sampled are skipped)
//   increment  left-multiplied twist xi = (omega, v):  p' = p + omega x p + v    =>  J_i = [ -[p_i]x^T grad ; grad ] = [ p_i x grad ; grad ]
//   gradient   grad = d psi / d p = the analytic derivative of the trilinear interpolant / voxel_size
//   step       (sum J J^T) xi = - sum J r   (6x6, Gaussian elimination with partial pivoting; a singular system ends the run)
//   update     R <- Rodrigues(omega) R,  t <- Rodrigues(omega) t + v
// trace rows [iters]: cost E before the step, number of valid points, |xi|.  Returns the iterations run (stops when
// |xi| < 1e-9 or the system is singular).
// ------------------------------------------------------------------------------------------------
int32_t orc_trilinear_grad(const orc_grid* g, const float* tsdf, const float* weight, const double xw[3], double* psi_out,
                           double grad_out[3]) {
  const long X = g->dims[0], Y = g->dims[1];
  double gc[3], f[3];
  long i0[3];
  for (int a = 0; a < 3; ++a) {
    gc[a] = (xw[a] - (double)g->origin[a]) / (double)g->voxel_size - 0.5;
    const double fl = std::floor(gc[a]);
    i0[a] = (long)fl;
    f[a] = gc[a] - fl;
  }
  if (!cell_ok(g, weight, i0[0], i0[1], i0[2])) return 0;
  double v[8];
  for (int c = 0; c < 8; ++c)
    v[c] = (double)tsdf[(i0[0] + (c & 1)) + X * ((i0[1] + ((c >> 1) & 1)) + Y * (i0[2] + ((c >> 2) & 1)))];
  double psi = 0, gx = 0, gy = 0, gz = 0;
  for (int c = 0; c < 8; ++c) {
    const int cx = c & 1, cy = (c >> 1) & 1, cz = (c >> 2) & 1;
    const double wx = cx ? f[0] : 1 - f[0], wy = cy ? f[1] : 1 - f[1], wz = cz ? f[2] : 1 - f[2];
    psi += wx * wy * wz * v[c];
    gx += (cx ? 1.0 : -1.0) * wy * wz * v[c];
    gy += wx * (cy ? 1.0 : -1.0) * wz * v[c];
    gz += wx * wy * (cz ? 1.0 : -1.0) * v[c];
  }
  *psi_out = psi;
  grad_out[0] = gx / (double)g->voxel_size; grad_out[1] = gy / (double)g->voxel_size; grad_out[2] = gz / (double)g->voxel_size;
  return 1;
}

struct orc_gn_row { double cost; int32_t n; int32_t pad; double step_norm; double A[36]; double b[6]; };

static bool solve6(double A[36], double b[6], double x[6]) {
  int n = 6;
  for (int c = 0; c < n; ++c) {
    int piv = c;
    for (int r = c + 1; r < n; ++r) if (std::fabs(A[6 * r + c]) > std::fabs(A[6 * piv + c])) piv = r;
    if (!(std::fabs(A[6 * piv + c]) > 1e-300)) return false;
    if (piv != c) { for (int k = 0; k < n; ++k) std::swap(A[6 * c + k], A[6 * piv + k]); std::swap(b[c], b[piv]); }
    for (int r = c + 1; r < n; ++r) {
      const double m = A[6 * r + c] / A[6 * c + c];
      for (int k = c; k < n; ++k) A[6 * r + k] -= m * A[6 * c + k];
      b[r] -= m * b[c];
    }
  }
  for (int r = n - 1; r >= 0; --r) {
    double sacc = b[r];
    for (int k = r + 1; k < n; ++k) sacc -= A[6 * r + k] * x[k];
    x[r] = sacc / A[6 * r + r];
  }
  return true;
}

static void rodrigues(const double w[3], double R[9]) {
  const double th = std::sqrt(w[0] * w[0] + w[1] * w[1] + w[2] * w[2]);
  double a, b;                                         // R = I + a [w]x + b [w]x^2
  if (th < 1e-8) { a = 1.0 - th * th / 6.0; b = 0.5 - th * th / 24.0; }
  else { a = std::sin(th) / th; b = (1.0 - std::cos(th)) / (th * th); }
  const double K[9] = {0, -w[2], w[1], w[2], 0, -w[0], -w[1], w[0], 0};
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      double k2 = 0;
      for (int k = 0; k < 3; ++k) k2 += K[3 * i + k] * K[3 * k + j];
      R[3 * i + j] = (i == j ? 1.0 : 0.0) + a * K[3 * i + j] + b * k2;
    }
}

int32_t orc_gn_track(const orc_grid* g, const float* tsdf, const float* weight, const float* points, int32_t M, double pose_io[12],
                     int32_t iters, orc_gn_row* rows) {
  double T[12];
  std::memcpy(T, pose_io, sizeof(T));
  int32_t k = 0;
  for (; k < iters; ++k) {
    double A[36] = {0}, b[6] = {0}, cost = 0;
    int32_t n = 0;
    for (int32_t i = 0; i < M; ++i) {
      if (points[4 * (size_t)i + 3] == 0.0f) continue;
      const double x[3] = {(double)points[4 * (size_t)i], (double)points[4 * (size_t)i + 1], (double)points[4 * (size_t)i + 2]};
      double p[3], psi, gr[3];
      for (int a = 0; a < 3; ++a) p[a] = T[4 * a] * x[0] + T[4 * a + 1] * x[1] + T[4 * a + 2] * x[2] + T[4 * a + 3];
      if (!orc_trilinear_grad(g, tsdf, weight, p, &psi, gr)) continue;
      const double J[6] = {p[1] * gr[2] - p[2] * gr[1], p[2] * gr[0] - p[0] * gr[2], p[0] * gr[1] - p[1] * gr[0], gr[0], gr[1], gr[2]};
      for (int r = 0; r < 6; ++r) { for (int c = 0; c < 6; ++c) A[6 * r + c] += J[r] * J[c]; b[r] += J[r] * psi; }
      cost += psi * psi; ++n;
    }
    if (rows) { rows[k].cost = cost; rows[k].n = n; rows[k].pad = 0; std::memcpy(rows[k].A, A, sizeof(A)); std::memcpy(rows[k].b, b, sizeof(b)); rows[k].step_norm = 0; }
    double rhs[6], xi[6];
    for (int r = 0; r < 6; ++r) rhs[r] = -b[r];
    if (n < 6 || !solve6(A, rhs, xi)) { ++k; break; }
    double Rw[9], Tn[12];
    rodrigues(xi, Rw);
    for (int i = 0; i < 3; ++i) {
      for (int j = 0; j < 3; ++j) Tn[4 * i + j] = Rw[3 * i] * T[j] + Rw[3 * i + 1] * T[4 + j] + Rw[3 * i + 2] * T[8 + j];
      Tn[4 * i + 3] = Rw[3 * i] * T[3] + Rw[3 * i + 1] * T[7] + Rw[3 * i + 2] * T[11] + xi[3 + i];
    }
    std::memcpy(T, Tn, sizeof(T));
    double nn = 0;
    for (int r = 0; r < 6; ++r) nn += xi[r] * xi[r];
    if (rows) rows[k].step_norm = std::sqrt(nn);
    if (std::sqrt(nn) < 1e-9) { ++k; break; }
  }
  std::memcpy(pose_io, T, sizeof(T));
  return k;
}

}  // extern "C"
