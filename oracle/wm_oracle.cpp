// =====================================================================================
// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// A plain, slow, scalar CPU restatement of what the Waymax closed-loop step computes
// (arXiv 2310.08710; citations are PAPER.md line numbers + section/equation, and the
// DESIGN.md reading numbers D1..D32 where the paper is silent).  Arithmetic is double
// precision; inputs and outputs are the float32 / uint8 / int32 arrays the CUDA library
// sees, and state is rounded to float32 at each step boundary.  It shares no code, header,
// table or helper with paper_2310_08710_b200/csrc; only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may call it.
//
// Parity pins (tests/test_oracle_*.py): every function below is pinned by closed forms,
// hand cases, brute force or invariants; none is "parity unpinned".
//
// The only loops that are parallel are `#pragma omp parallel for` over scenarios b
// (scenarios are independent); nothing else is blocked, fused or
// reordered.
// =====================================================================================
#include <algorithm>
#include <cfloat>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

struct orc_traj {            // [B][T][A] each, time-major
  int32_t B, A, T;
  float *x, *y, *yaw, *vel_x, *vel_y, *length, *width;
  uint8_t* valid;
};
struct orc_roadgraph {       // [B][R] each
  int32_t B, R;
  float *x, *y, *dir_x, *dir_y;
  int32_t *type, *id;
  uint8_t* valid;
};

enum { ORC_DYN_BICYCLE = 0, ORC_DYN_DELTA_LOCAL = 1, ORC_DYN_DELTA_GLOBAL = 2 };
enum { ORC_TYPE_ROAD_EDGE = 2 };

static inline size_t row(const orc_traj* tr, int b, int t) {
  return ((size_t)b * tr->T + t) * tr->A;
}

// -------------------------------------------------------------------------------------
// O1/O2 + D8/D9: one transition, row t -> row t+1.
//   InvertibleBicycle: PAPER.md L339-L350 (Appendix A.1, Eq. 2), literal: the position uses
//     the velocity components, the acceleration term uses the yaw.
//   DeltaLocal: PAPER.md L324-L333 (Eq. 1) after rotating the body-frame delta by yaw (D2).
//   DeltaGlobal: Eq. 1 literally, the delta is in the world frame.
//   Action clipping to +-max_accel / +-max_curvature when the limit is > 0 (D7; limits
//     6 m/s^2, 0.3 1/m from L104).
//   use_dyn = action_valid && sim.valid[t]; otherwise row t+1 <- log row t+1 (D8, L164).
//   Controlled: valid'=1, length/width carried over (D9). No yaw wrapping (D5), no speed
//   clamp (D6).
// action: [B][C][A] with batch stride `act_stride_b` floats (C=2: a,kappa; C=3: dx,dy,dyaw).
// -------------------------------------------------------------------------------------
void orc_step(const orc_traj* log, orc_traj* sim, int32_t t, int32_t dynamics, double dt,
              double max_accel, double max_curvature, const float* action,
              int64_t act_stride_b, const uint8_t* action_valid, int64_t av_stride_b) {
  const int B = sim->B, A = sim->A;
#pragma omp parallel for schedule(static)
  for (int b = 0; b < B; ++b) {
    const size_t r0 = row(sim, b, t), r1 = row(sim, b, t + 1), l1 = row(log, b, t + 1);
    const float* act = action + (size_t)b * act_stride_b;
    const uint8_t* av = action_valid + (size_t)b * av_stride_b;
    for (int a = 0; a < A; ++a) {
      const bool use_dyn = av[a] != 0 && sim->valid[r0 + a] != 0;
      if (!use_dyn) {
        sim->x[r1 + a] = log->x[l1 + a];
        sim->y[r1 + a] = log->y[l1 + a];
        sim->yaw[r1 + a] = log->yaw[l1 + a];
        sim->vel_x[r1 + a] = log->vel_x[l1 + a];
        sim->vel_y[r1 + a] = log->vel_y[l1 + a];
        sim->length[r1 + a] = log->length[l1 + a];
        sim->width[r1 + a] = log->width[l1 + a];
        sim->valid[r1 + a] = log->valid[l1 + a];
        continue;
      }
      const double x = sim->x[r0 + a], y = sim->y[r0 + a], th = sim->yaw[r0 + a];
      const double vx = sim->vel_x[r0 + a], vy = sim->vel_y[r0 + a];
      double xn, yn, thn, vxn, vyn;
      if (dynamics == ORC_DYN_BICYCLE) {
        double acc = act[0 * A + a], kappa = act[1 * A + a];
        if (max_accel > 0) acc = std::min(std::max(acc, -max_accel), max_accel);
        if (max_curvature > 0) kappa = std::min(std::max(kappa, -max_curvature), max_curvature);
        const double v = std::sqrt(vx * vx + vy * vy);
        xn = x + vx * dt + 0.5 * acc * std::cos(th) * dt * dt;       // Eq. 2
        yn = y + vy * dt + 0.5 * acc * std::sin(th) * dt * dt;       // L341
        thn = th + kappa * (v * dt + 0.5 * acc * dt * dt);           // L343
        const double vn = v + acc * dt;                              // L345
        vxn = vn * std::cos(thn);                                    // L347
        vyn = vn * std::sin(thn);                                    // L349
      } else {
        const double dx = act[0 * A + a], dy = act[1 * A + a], dyaw = act[2 * A + a];
        // DeltaGlobal: Eq. 1 literally (world-frame delta); DeltaLocal: the body-frame delta rotated by yaw (D2)
        const double c = dynamics == ORC_DYN_DELTA_GLOBAL ? 1.0 : std::cos(th), s = dynamics == ORC_DYN_DELTA_GLOBAL ? 0.0 : std::sin(th);
        xn = x + c * dx - s * dy;                                    // Eq. 1, world delta
        yn = y + s * dx + c * dy;                                    // L326
        thn = th + dyaw;                                             // L328
        // Eq. 1: v' = (x'-x)/dt, evaluated on the float32 state that is stored.
        const double xs = (double)(float)xn, ys = (double)(float)yn;
        vxn = (xs - x) / dt;
        vyn = (ys - y) / dt;
      }
      sim->x[r1 + a] = (float)xn;
      sim->y[r1 + a] = (float)yn;
      sim->yaw[r1 + a] = (float)thn;
      sim->vel_x[r1 + a] = (float)vxn;
      sim->vel_y[r1 + a] = (float)vyn;
      sim->length[r1 + a] = sim->length[r0 + a];
      sim->width[r1 + a] = sim->width[r0 + a];
      sim->valid[r1 + a] = 1;
    }
  }
}

// a0 (L122, L78): sim[0..history-1] <- log[0..history-1]; later rows invalid and zero.
void orc_reset(const orc_traj* log, orc_traj* sim, int32_t history) {
  const int B = sim->B, A = sim->A, T = sim->T;
  for (int b = 0; b < B; ++b)
    for (int t = 0; t < T; ++t) {
      const size_t r = row(sim, b, t);
      for (int a = 0; a < A; ++a) {
        const bool c = t < history;
        sim->x[r + a] = c ? log->x[r + a] : 0.f;
        sim->y[r + a] = c ? log->y[r + a] : 0.f;
        sim->yaw[r + a] = c ? log->yaw[r + a] : 0.f;
        sim->vel_x[r + a] = c ? log->vel_x[r + a] : 0.f;
        sim->vel_y[r + a] = c ? log->vel_y[r + a] : 0.f;
        sim->length[r + a] = c ? log->length[r + a] : 0.f;
        sim->width[r + a] = c ? log->width[r + a] : 0.f;
        sim->valid[r + a] = c ? log->valid[r + a] : 0;
      }
    }
}

// -------------------------------------------------------------------------------------
// O3 overlap (collision metric): two oriented rectangles intersect with
// positive area iff no edge-normal axis separates them.
//   gap(i,j) = max over the 4 edge normals u of |u.(c_j-c_i)| - (r_i(u)+r_j(u)),
//   r(u) = (L/2)|u.f| + (W/2)|u.s|;  overlap = valid_i && valid_j && i!=j && gap<0 (D12,D13)
// Outputs: gap [B][A][A] double (may be NULL; +inf where not evaluated), pair [B][A][A]
// uint8 (may be NULL), flag [B][A] uint8 (row OR).
// -------------------------------------------------------------------------------------
void orc_overlap(const orc_traj* sim, int32_t t, double* gap, uint8_t* pair, uint8_t* flag) {
  const int B = sim->B, A = sim->A;
#pragma omp parallel for schedule(static)
  for (int b = 0; b < B; ++b) {
    const size_t r = row(sim, b, t);
    for (int i = 0; i < A; ++i) {
      uint8_t any = 0;
      for (int j = 0; j < A; ++j) {
        double g = INFINITY;
        uint8_t ov = 0;
        if (i != j && sim->valid[r + i] && sim->valid[r + j]) {
          const double ci[2] = {sim->x[r + i], sim->y[r + i]}, cj[2] = {sim->x[r + j], sim->y[r + j]};
          const double thi = sim->yaw[r + i], thj = sim->yaw[r + j];
          const double fi[2] = {std::cos(thi), std::sin(thi)}, si[2] = {-std::sin(thi), std::cos(thi)};
          const double fj[2] = {std::cos(thj), std::sin(thj)}, sj[2] = {-std::sin(thj), std::cos(thj)};
          const double hli = 0.5 * sim->length[r + i], hwi = 0.5 * sim->width[r + i];
          const double hlj = 0.5 * sim->length[r + j], hwj = 0.5 * sim->width[r + j];
          const double d[2] = {cj[0] - ci[0], cj[1] - ci[1]};
          const double* axes[4] = {fi, si, fj, sj};
          g = -INFINITY;
          for (int k = 0; k < 4; ++k) {
            const double* u = axes[k];
            const double ri = hli * std::fabs(u[0] * fi[0] + u[1] * fi[1]) + hwi * std::fabs(u[0] * si[0] + u[1] * si[1]);
            const double rj = hlj * std::fabs(u[0] * fj[0] + u[1] * fj[1]) + hwj * std::fabs(u[0] * sj[0] + u[1] * sj[1]);
            const double sep = std::fabs(u[0] * d[0] + u[1] * d[1]) - (ri + rj);
            g = std::max(g, sep);
          }
          ov = g < 0.0;
        }
        if (gap) gap[((size_t)b * A + i) * A + j] = g;
        if (pair) pair[((size_t)b * A + i) * A + j] = ov;
        any |= ov;
      }
      flag[(size_t)b * A + i] = any;
    }
  }
}

// -------------------------------------------------------------------------------------
// O4 offroad (readings D14-D20).
// Segments: consecutive array entries (i,i+1), both valid, both ROAD_EDGE, same id; a valid
// road-edge point that starts no segment and ends none is a zero-length segment.  The sign
// direction is the segment vector e, or the stored dir when e = 0 (D16).
// Per corner q (corner order: 0 front-left, 1 front-right, 2 rear-right, 3 rear-left):
//   t* = clamp(((q-p0).e)/(e.e),0,1); closest = p0 | p1 | p0+t*e; d = |q-closest|;
//   winner = min d, exact ties -> lower index (D17); side = e x (q-p0);
//   sd = side>0 ? -d : +d (left of the oriented edge = on-road = negative).
// Agent value = max over corners; flag = valid && sd_max > 0 (D18, D19).  No segments:
// sd = -FLT_MAX, flag 0 (D20).  Invalid agents: outputs 0 (D10).
// Ambiguity (P15) per corner: d < band, lateral |side|/|e| < band, or a segment of the
// opposite sign within band of the winning distance.
// Outputs: sd [B][A], corner_sd [B][4][A] (may be NULL), flag [B][A], ambig [B][4][A] (NULL ok),
// win_seg [B][4][A] int32 = first-point index of the winning segment (NULL ok).
// -------------------------------------------------------------------------------------
struct OrcSeg { double p0x, p0y, p1x, p1y, sx, sy; int32_t src; };

static void build_segments(const orc_roadgraph* rg, int b, std::vector<OrcSeg>& segs) {
  const int R = rg->R;
  const size_t o = (size_t)b * R;
  segs.clear();
  auto edge = [&](int i) { return rg->valid[o + i] != 0 && rg->type[o + i] == ORC_TYPE_ROAD_EDGE; };
  auto starts = [&](int i) { return i + 1 < R && edge(i) && edge(i + 1) && rg->id[o + i] == rg->id[o + i + 1]; };
  for (int i = 0; i < R; ++i) {
    const bool s = starts(i);
    const bool iso = edge(i) && !s && !(i > 0 && starts(i - 1));
    if (!s && !iso) continue;
    OrcSeg g;
    g.p0x = rg->x[o + i]; g.p0y = rg->y[o + i];
    if (s) { g.p1x = rg->x[o + i + 1]; g.p1y = rg->y[o + i + 1]; } else { g.p1x = g.p0x; g.p1y = g.p0y; }
    const double ex = g.p1x - g.p0x, ey = g.p1y - g.p0y;
    if (ex * ex + ey * ey > 0.0) { g.sx = ex; g.sy = ey; } else { g.sx = rg->dir_x[o + i]; g.sy = rg->dir_y[o + i]; }
    g.src = i;
    segs.push_back(g);
  }
}

int32_t orc_count_segments(const orc_roadgraph* rg, int32_t b) {
  std::vector<OrcSeg> segs; build_segments(rg, b, segs); return (int32_t)segs.size();
}

void orc_offroad(const orc_traj* sim, int32_t t, const orc_roadgraph* rg, double band, float* sd_out,
                 float* corner_sd, uint8_t* flag, uint8_t* ambig, int32_t* win_seg) {
  const int B = sim->B, A = sim->A;
#pragma omp parallel for schedule(dynamic, 1)
  for (int b = 0; b < B; ++b) {
    std::vector<OrcSeg> segs;
    build_segments(rg, b, segs);
    const size_t r = row(sim, b, t);
    for (int a = 0; a < A; ++a) {
      const size_t oa = (size_t)b * A + a;
      if (!sim->valid[r + a]) {
        sd_out[oa] = 0.f; flag[oa] = 0;
        for (int k = 0; k < 4; ++k) {
          const size_t oc = ((size_t)b * 4 + k) * A + a;
          if (corner_sd) corner_sd[oc] = 0.f;
          if (ambig) ambig[oc] = 0;
          if (win_seg) win_seg[oc] = -1;
        }
        continue;
      }
      const double cx = sim->x[r + a], cy = sim->y[r + a], th = sim->yaw[r + a];
      const double hl = 0.5 * sim->length[r + a], hw = 0.5 * sim->width[r + a];
      const double fx = std::cos(th), fy = std::sin(th), sx = -std::sin(th), sy = std::cos(th);
      const double sl[4] = {+1, +1, -1, -1}, sw[4] = {+1, -1, -1, +1};  // FL, FR, RR, RL
      double sd_max = -DBL_MAX;
      for (int k = 0; k < 4; ++k) {
        const double qx = cx + sl[k] * hl * fx + sw[k] * hw * sx;
        const double qy = cy + sl[k] * hl * fy + sw[k] * hw * sy;
        double best = INFINITY, best_side = 0, best_snorm = 1; int best_i = -1;
        double best_pos = INFINITY, best_neg = INFINITY;   // min d among side>0 / side<=0 segments
        for (size_t i = 0; i < segs.size(); ++i) {
          const OrcSeg& g = segs[i];
          const double ex = g.p1x - g.p0x, ey = g.p1y - g.p0y, ee = ex * ex + ey * ey;
          const double wx = qx - g.p0x, wy = qy - g.p0y;
          double px = g.p0x, py = g.p0y;
          if (ee > 0.0) {
            double ts = (wx * ex + wy * ey) / ee;
            ts = std::min(std::max(ts, 0.0), 1.0);
            if (ts <= 0.0) { px = g.p0x; py = g.p0y; }
            else if (ts >= 1.0) { px = g.p1x; py = g.p1y; }
            else { px = g.p0x + ts * ex; py = g.p0y + ts * ey; }
          }
          const double d = std::sqrt((qx - px) * (qx - px) + (qy - py) * (qy - py));
          const double side = g.sx * wy - g.sy * wx;
          if (side > 0) best_pos = std::min(best_pos, d); else best_neg = std::min(best_neg, d);
          if (d < best) { best = d; best_side = side; best_snorm = std::sqrt(g.sx * g.sx + g.sy * g.sy); best_i = g.src; }
        }
        double sd; uint8_t amb = 0;
        if (best_i < 0) { sd = -(double)FLT_MAX; }
        else {
          sd = best_side > 0 ? -best : best;
          const double opp = best_side > 0 ? best_neg : best_pos;
          const double lateral = best_snorm > 0 ? std::fabs(best_side) / best_snorm : 0.0;
          amb = (best < band) || (lateral < band) || (opp - best < band);
        }
        const size_t oc = ((size_t)b * 4 + k) * A + a;
        if (corner_sd) corner_sd[oc] = (float)sd;
        if (ambig) ambig[oc] = amb;
        if (win_seg) win_seg[oc] = best_i;
        sd_max = std::max(sd_max, sd);
      }
      sd_out[oa] = (float)sd_max;
      flag[oa] = sd_max > 0.0;
    }
  }
}

// -------------------------------------------------------------------------------------
// O5 log divergence (displacement error): L2 distance between simulated and
// logged XY at the same timestep; valid iff both valid, else 0.
// -------------------------------------------------------------------------------------
void orc_log_divergence(const orc_traj* log, const orc_traj* sim, int32_t t, float* dist, uint8_t* valid) {
  const int B = sim->B, A = sim->A;
  for (int b = 0; b < B; ++b) {
    const size_t r = row(sim, b, t), l = row(log, b, t);
    for (int a = 0; a < A; ++a) {
      const bool v = sim->valid[r + a] && log->valid[l + a];
      double d = 0;
      if (v) {
        const double dx = (double)sim->x[r + a] - log->x[l + a], dy = (double)sim->y[r + a] - log->y[l + a];
        d = std::sqrt(dx * dx + dy * dy);
      }
      dist[(size_t)b * A + a] = (float)d;
      valid[(size_t)b * A + a] = v;
    }
  }
}

// -------------------------------------------------------------------------------------
// O6 observation, history part (D22): for each ego e valid at t and every
// agent a, steps t-H+1..t: p' = R(-yaw_e)(p - p_e), yaw' = wrap(yaw - yaw_e) to [-pi,pi),
// v' = R(-yaw_e) v, length/width copied; valid' = valid[a,h] && valid[e,t]; invalid -> 0.
// hist [B][E][H][7][A] (x,y,yaw,vx,vy,length,width), hist_valid [B][E][H][A].
// -------------------------------------------------------------------------------------
static double wrap_pi(double a) {
  const double two_pi = 2.0 * M_PI;
  double w = std::fmod(a + M_PI, two_pi);
  if (w < 0) w += two_pi;
  return w - M_PI;
}

void orc_observe_history(const orc_traj* sim, int32_t t, int32_t H, float* hist, uint8_t* hist_valid) {
  const int B = sim->B, A = sim->A;
#pragma omp parallel for schedule(static)
  for (int b = 0; b < B; ++b) {
    const size_t rt = row(sim, b, t);
    for (int e = 0; e < A; ++e) {
      const bool ev = sim->valid[rt + e] != 0;
      const double ex = ev ? sim->x[rt + e] : 0, ey = ev ? sim->y[rt + e] : 0, eth = ev ? sim->yaw[rt + e] : 0;
      const double c = std::cos(eth), s = std::sin(eth);
      for (int h = 0; h < H; ++h) {
        const size_t rh = row(sim, b, t - H + 1 + h);
        for (int a = 0; a < A; ++a) {
          const bool v = ev && sim->valid[rh + a] != 0;
          double o[7] = {0, 0, 0, 0, 0, 0, 0};
          if (v) {
            const double dx = sim->x[rh + a] - ex, dy = sim->y[rh + a] - ey;
            o[0] = c * dx + s * dy;
            o[1] = -s * dx + c * dy;
            o[2] = wrap_pi((double)sim->yaw[rh + a] - eth);
            const double vx = sim->vel_x[rh + a], vy = sim->vel_y[rh + a];
            o[3] = c * vx + s * vy;
            o[4] = -s * vx + c * vy;
            o[5] = sim->length[rh + a];
            o[6] = sim->width[rh + a];
          }
          const size_t base = ((((size_t)b * A + e) * H + h) * 7) * A + a;
          for (int f = 0; f < 7; ++f) hist[base + (size_t)f * A] = (float)o[f];
          hist_valid[(((size_t)b * A + e) * H + h) * A + a] = v;
        }
      }
    }
  }
}

// -------------------------------------------------------------------------------------
// O7 observation, roadgraph part ("sub-samples the roadgraph via distance";
// D23-D25): for each ego valid at t, the k valid roadgraph points nearest the ego centre,
// ties -> lower index, emitted in ascending index order (order = 0, D24) or by ascending
// (distance key, index) — the sorted-by-distance variant of SURVEY 8(f)(4), D44 (order = 1) —, padded with -1.
// The integer decision (which points) is taken in float32, the kernel's precision:
//   key = fma(dy, dy, dx*dx) with dx = fl(px-ex), dy = fl(py-ey), round-to-nearest
// (DESIGN.md R-topk).  Features are computed in double: p' = R(-yaw_e)(p-p_e),
// dir' = R(-yaw_e) dir.  Also returns kth_key [B][E] = float32 key of the k-th selected point
// (NaN if fewer than k valid points) for the band report.
// rg_index [B][E][k], rg_feat [B][E][4][k] (x,y,dir_x,dir_y), rg_type [B][E][k].
// -------------------------------------------------------------------------------------
void orc_observe_topk(const orc_traj* sim, const orc_roadgraph* rg, int32_t t, int32_t k, int32_t order,
                      int32_t* rg_index, float* rg_feat, int32_t* rg_type, float* kth_key) {
  const int B = sim->B, A = sim->A, R = rg->R;
#pragma omp parallel for schedule(dynamic, 1)
  for (int b = 0; b < B; ++b) {
    const size_t rt = row(sim, b, t), o = (size_t)b * R;
    std::vector<std::pair<float, int32_t>> keys;
    std::vector<int32_t> sel;
    for (int e = 0; e < A; ++e) {
      int32_t* oi = rg_index + ((size_t)b * A + e) * k;
      float* of = rg_feat + ((size_t)b * A + e) * 4 * k;
      int32_t* ot = rg_type + ((size_t)b * A + e) * k;
      for (int j = 0; j < k; ++j) { oi[j] = -1; ot[j] = 0; of[j] = of[k + j] = of[2 * k + j] = of[3 * k + j] = 0.f; }
      if (kth_key) kth_key[(size_t)b * A + e] = NAN;
      if (!sim->valid[rt + e]) continue;
      const float exf = sim->x[rt + e], eyf = sim->y[rt + e];
      keys.clear();
      for (int i = 0; i < R; ++i) {
        if (!rg->valid[o + i]) continue;
        const float dx = rg->x[o + i] - exf, dy = rg->y[o + i] - eyf;
        const float key = std::fmaf(dy, dy, dx * dx);
        keys.emplace_back(key, i);
      }
      std::sort(keys.begin(), keys.end());      // lexicographic (key, index)
      const int n = std::min<int>(k, (int)keys.size());
      sel.clear();
      for (int j = 0; j < n; ++j) sel.push_back(keys[j].second);
      if (order == 0) std::sort(sel.begin(), sel.end());        // ascending index (D24); order 1: by (distance key, index), D44
      if (kth_key && (int)keys.size() >= k && k > 0) kth_key[(size_t)b * A + e] = keys[k - 1].first;
      const double ex = exf, ey = eyf, eth = sim->yaw[rt + e];
      const double c = std::cos(eth), s = std::sin(eth);
      for (int j = 0; j < n; ++j) {
        const int i = sel[j];
        const double dx = rg->x[o + i] - ex, dy = rg->y[o + i] - ey;
        const double ux = rg->dir_x[o + i], uy = rg->dir_y[o + i];
        oi[j] = i;
        of[0 * k + j] = (float)(c * dx + s * dy);
        of[1 * k + j] = (float)(-s * dx + c * dy);
        of[2 * k + j] = (float)(c * ux + s * uy);
        of[3 * k + j] = (float)(-s * ux + c * uy);
        ot[j] = rg->type[o + i];
      }
    }
  }
}

// -------------------------------------------------------------------------------------
// O8 rollout (D11, D21): n_steps x (O1/O2 -> O3, O4, O5 on row t+1).
// Per-step rows [B][n_steps][A]; aggregates [B][A]: any-overlap, any-offroad,
// ADE = sum of valid distances / count (0 if count 0).  actions [B][n_steps][C][A],
// action_valid [B][n_steps][A].  Any output pointer may be NULL.
// -------------------------------------------------------------------------------------
void orc_rollout(const orc_traj* log, orc_traj* sim, const orc_roadgraph* rg, int32_t t0, int32_t n_steps,
                 int32_t dynamics, double dt, double max_accel, double max_curvature,
                 const float* actions, const uint8_t* action_valid, double band,
                 uint8_t* overlap, uint8_t* offroad, float* offroad_dist, float* log_div,
                 uint8_t* any_overlap, uint8_t* any_offroad, float* ade) {
  const int B = sim->B, A = sim->A;
  const int C = dynamics == ORC_DYN_BICYCLE ? 2 : 3;
  const size_t BA = (size_t)B * A;
  std::vector<uint8_t> f_ov(BA), f_off(BA), v_ld(BA);
  std::vector<float> sd(BA), ld(BA);
  std::vector<double> sum(BA, 0.0);
  std::vector<int32_t> cnt(BA, 0);
  if (any_overlap) std::memset(any_overlap, 0, BA);
  if (any_offroad) std::memset(any_offroad, 0, BA);
  for (int s = 0; s < n_steps; ++s) {
    const int t = t0 + s;
    orc_step(log, sim, t, dynamics, dt, max_accel, max_curvature, actions + (size_t)s * C * A,
             (int64_t)n_steps * C * A, action_valid + (size_t)s * A, (int64_t)n_steps * A);
    orc_overlap(sim, t + 1, nullptr, nullptr, f_ov.data());
    orc_offroad(sim, t + 1, rg, band, sd.data(), nullptr, f_off.data(), nullptr, nullptr);
    orc_log_divergence(log, sim, t + 1, ld.data(), v_ld.data());
    for (int b = 0; b < B; ++b)
      for (int a = 0; a < A; ++a) {
        const size_t i = (size_t)b * A + a, o = ((size_t)b * n_steps + s) * A + a;
        if (overlap) overlap[o] = f_ov[i];
        if (offroad) offroad[o] = f_off[i];
        if (offroad_dist) offroad_dist[o] = sd[i];
        if (log_div) log_div[o] = ld[i];
        if (any_overlap) any_overlap[i] |= f_ov[i];
        if (any_offroad) any_offroad[i] |= f_off[i];
        if (v_ld[i]) { sum[i] += ld[i]; cnt[i] += 1; }
      }
  }
  if (ade)
    for (size_t i = 0; i < BA; ++i) ade[i] = cnt[i] ? (float)(sum[i] / cnt[i]) : 0.f;
}

// -------------------------------------------------------------------------------------
// O9 expert actor = inverse kinematics on two consecutive rows ("Expert";
// L335 delta inverse; L352-L359 Eq. 3 bicycle inverse).  Steps s = 0..n_steps-1 use rows
// t+s and t+s+1 of `tr`.  Output action [B][n_steps][C][A], valid [B][n_steps][A] = both rows
// valid; invalid -> action 0.
//   bicycle (Eq. 3):  a = (v' - v) / dt,  v = sqrt(vx^2 + vy^2)
//                     kappa = wrap(atan2(vy', vx') - theta) / (v dt + a dt^2 / 2)
//     D4: the heading is atan2(v_y', v_x') (the paper's "arctan v_x'/v_y'" is garbled);
//     D32: the heading difference is wrapped into [-pi, pi) (yaw is not wrapped in step, D5);
//     D31: kappa = 0 when the float32 speeds v and v' are both exactly 0 (denominator 0).
//   delta (L335) in the body frame of row t+s (D2): (dx, dy) = R(-theta) (p' - p), dyaw = theta' - theta.
// `kden` (may be NULL, bicycle only): the denominator of kappa, for the test tolerances.
// -------------------------------------------------------------------------------------
static double orc_wrap_pi(double a) {
  const double two_pi = 6.283185307179586476925286766559;
  a = std::fmod(a + 3.14159265358979323846, two_pi);
  if (a < 0) a += two_pi;
  return a - 3.14159265358979323846;
}

static void inverse_bicycle(const orc_traj* tr, size_t i0, size_t i1, double dt, double* a_out, double* k_out, double* den_out) {
  const double vx = tr->vel_x[i0], vy = tr->vel_y[i0], vx1 = tr->vel_x[i1], vy1 = tr->vel_y[i1];
  const double v = std::sqrt(vx * vx + vy * vy), v1 = std::sqrt(vx1 * vx1 + vy1 * vy1);
  const double a = (v1 - v) / dt;                                   // Eq. 3
  const double den = v * dt + 0.5 * a * dt * dt;                    // L358
  double kappa = 0.0;
  if (!(v == 0.0 && v1 == 0.0)) kappa = orc_wrap_pi(std::atan2(vy1, vx1) - (double)tr->yaw[i0]) / den;   // D4, D31, D32
  *a_out = a; *k_out = kappa; *den_out = den;
}

void orc_expert_actions(const orc_traj* tr, int32_t t, int32_t n_steps, int32_t dynamics, double dt, float* action,
                        uint8_t* valid, double* kden) {
  const int B = tr->B, A = tr->A;
  const int C = dynamics == ORC_DYN_BICYCLE ? 2 : 3;
#pragma omp parallel for schedule(static)
  for (int b = 0; b < B; ++b)
    for (int s = 0; s < n_steps; ++s)
      for (int a = 0; a < A; ++a) {
        const size_t i0 = row(tr, b, t + s) + a, i1 = row(tr, b, t + s + 1) + a;
        const size_t o = (((size_t)b * n_steps + s) * C) * A + a, ov = ((size_t)b * n_steps + s) * A + a;
        const bool v = tr->valid[i0] != 0 && tr->valid[i1] != 0;
        valid[ov] = (uint8_t)v;
        for (int c = 0; c < C; ++c) action[o + (size_t)c * A] = 0.f;
        if (kden) kden[ov] = 0.0;
        if (!v) continue;
        if (dynamics == ORC_DYN_BICYCLE) {
          double acc, kap, den;
          inverse_bicycle(tr, i0, i1, dt, &acc, &kap, &den);
          action[o] = (float)acc; action[o + A] = (float)kap;
          if (kden) kden[ov] = den;
        } else {
          const double th = tr->yaw[i0];
          const double cs = dynamics == ORC_DYN_DELTA_GLOBAL ? 1.0 : std::cos(th), sn = dynamics == ORC_DYN_DELTA_GLOBAL ? 0.0 : std::sin(th);
          const double Dx = (double)tr->x[i1] - (double)tr->x[i0], Dy = (double)tr->y[i1] - (double)tr->y[i0];   // L335
          action[o] = (float)(cs * Dx + sn * Dy);                   // body frame (D2); DeltaGlobal: (Dx, Dy) itself
          action[o + A] = (float)(-sn * Dx + cs * Dy);
          action[o + 2 * (size_t)A] = (float)((double)tr->yaw[i1] - th);
        }
      }
}

// -------------------------------------------------------------------------------------
// O10 kinematic infeasibility: Eq. 3 on rows t+s-1 -> t+s, s = 0..n_steps-1;
// flag = |a| > max_accel or |kappa| > max_curvature (6 m/s^2, 0.3 1/m), strictly.
// Outputs [B][n_steps][A]; valid = both rows valid, otherwise 0 / flag 0.
// -------------------------------------------------------------------------------------
void orc_kinematic(const orc_traj* tr, int32_t t, int32_t n_steps, double dt, double max_accel, double max_curvature,
                   float* accel, float* curvature, double* kden, uint8_t* flag, uint8_t* valid) {
  const int B = tr->B, A = tr->A;
#pragma omp parallel for schedule(static)
  for (int b = 0; b < B; ++b)
    for (int s = 0; s < n_steps; ++s)
      for (int a = 0; a < A; ++a) {
        const size_t i0 = row(tr, b, t + s - 1) + a, i1 = row(tr, b, t + s) + a;
        const size_t o = ((size_t)b * n_steps + s) * A + a;
        const bool v = tr->valid[i0] != 0 && tr->valid[i1] != 0;
        double acc = 0.0, kap = 0.0, den = 0.0;
        if (v) inverse_bicycle(tr, i0, i1, dt, &acc, &kap, &den);
        accel[o] = (float)acc; curvature[o] = (float)kap;
        if (kden) kden[o] = den;
        flag[o] = (uint8_t)(v && (std::fabs(acc) > max_accel || std::fabs(kap) > max_curvature));
        valid[o] = (uint8_t)v;
      }
}

// -------------------------------------------------------------------------------------
// O11 route progress ratio: "associates the vehicle's position to the closest
// point x(t) in an on-route path ... distance along the path from the start of the path to
// x(t), d_x(t) ... ratio = (d_x(t) - d_p) / (d_q - d_p), where d_p and d_q are the distances along
// the path to the initial and final positions of the vehicle's logged trajectory ... could be
// greater than 1".  One on-route path per agent: points [B][A][P] with their arc length (an
// input, as in the paper's path structure) and validity.
//   D33: closest POINT (not segment) among the valid path points, ties -> lower index; the
//        comparison key is the float32 value fma(dy, dy, dx*dx) (the kernel's precision, as for
//        the top-k: a floating-point value that decides an index);
//   D34: initial / final logged position = first / last VALID logged row of the agent;
//   D35: valid = sim valid at t, some valid path point, some valid logged row, d_q != d_p;
//        otherwise ratio 0, valid 0.
// closest (may be NULL): [B][3][A] indices of the closest points to (sim, log first, log last).
// -------------------------------------------------------------------------------------
struct orc_paths { int32_t B, A, P; float *x, *y, *arc_len; uint8_t* valid; };

static int closest_path_point(const orc_paths* pa, int b, int a, float qx, float qy) {
  const size_t o = ((size_t)b * pa->A + a) * pa->P;
  int best = -1;
  float bk = 0.f;
  for (int i = 0; i < pa->P; ++i) {
    if (!pa->valid[o + i]) continue;
    const float dx = pa->x[o + i] - qx, dy = pa->y[o + i] - qy;        // float32 on purpose (D33)
    const float key = std::fmaf(dy, dy, dx * dx);
    if (best < 0 || key < bk) { best = i; bk = key; }                   // strict '<': ties -> lower index
  }
  return best;
}

void orc_route_progress(const orc_traj* log, const orc_traj* sim, int32_t t, const orc_paths* pa, float* ratio,
                        uint8_t* valid, int32_t* closest) {
  const int B = sim->B, A = sim->A, T = sim->T;
#pragma omp parallel for schedule(static)
  for (int b = 0; b < B; ++b)
    for (int a = 0; a < A; ++a) {
      const size_t o = (size_t)b * A + a;
      ratio[o] = 0.f; valid[o] = 0;
      if (closest) for (int c = 0; c < 3; ++c) closest[((size_t)b * 3 + c) * A + a] = -1;
      int tf = -1, tl = -1;                                              // D34
      for (int k = 0; k < T; ++k) if (log->valid[row(log, b, k) + a]) { if (tf < 0) tf = k; tl = k; }
      const size_t rs = row(sim, b, t) + a;
      if (!sim->valid[rs] || tf < 0) continue;
      const int ix = closest_path_point(pa, b, a, sim->x[rs], sim->y[rs]);
      if (ix < 0) continue;
      const int ip = closest_path_point(pa, b, a, log->x[row(log, b, tf) + a], log->y[row(log, b, tf) + a]);
      const int iq = closest_path_point(pa, b, a, log->x[row(log, b, tl) + a], log->y[row(log, b, tl) + a]);
      if (closest) { closest[((size_t)b * 3 + 0) * A + a] = ix; closest[((size_t)b * 3 + 1) * A + a] = ip; closest[((size_t)b * 3 + 2) * A + a] = iq; }
      const size_t po = ((size_t)b * pa->A + a) * pa->P;
      const double dxp = pa->arc_len[po + ix], dp = pa->arc_len[po + ip], dq = pa->arc_len[po + iq];
      if (dq == dp) continue;                                            // D35
      ratio[o] = (float)((dxp - dp) / (dq - dp));                        // L96
      valid[o] = 1;
    }
}

// -------------------------------------------------------------------------------------
// O12 off-route metric: "If the vehicle is sufficiently closer to an off-route path
// than on-route path or it is far enough away from an on-route path, it is considered off-route."
// The two thresholds are not in the paper: they are arguments (D36).  d_on / d_off = distance from
// the agent's position at row t to the closest valid point of its on-route / off-route path
// (closest POINT, float32 key and float32 square root as in D33; +inf without an off-route point);
//   flag = d_on > max_dist  ||  d_off + margin < d_on
// for agents valid at t that have an on-route path point; otherwise flag 0, dist 0.
// off may be NULL (no off-route paths).  dist_on [B][A] (float32), flag [B][A].
// -------------------------------------------------------------------------------------
static float closest_path_dist(const orc_paths* pa, int b, int a, float qx, float qy, bool* found) {
  const int i = closest_path_point(pa, b, a, qx, qy);
  *found = i >= 0;
  if (i < 0) return INFINITY;
  const size_t o = ((size_t)b * pa->A + a) * pa->P + i;
  const float dx = pa->x[o] - qx, dy = pa->y[o] - qy;                  // float32 on purpose (D33 / D36)
  return std::sqrt(std::fmaf(dy, dy, dx * dx));
}

void orc_offroute(const orc_traj* sim, int32_t t, const orc_paths* on, const orc_paths* off, float max_dist, float margin,
                  float* dist_on, uint8_t* flag) {
  const int B = sim->B, A = sim->A;
#pragma omp parallel for schedule(static)
  for (int b = 0; b < B; ++b)
    for (int a = 0; a < A; ++a) {
      const size_t o = (size_t)b * A + a, rs = row(sim, b, t) + a;
      dist_on[o] = 0.f; flag[o] = 0;
      if (!sim->valid[rs]) continue;
      bool f_on = false, f_off = false;
      const float d_on = closest_path_dist(on, b, a, sim->x[rs], sim->y[rs], &f_on);
      if (!f_on) continue;
      const float d_off = off ? closest_path_dist(off, b, a, sim->x[rs], sim->y[rs], &f_off) : INFINITY;
      dist_on[o] = d_on;
      flag[o] = (uint8_t)(d_on > max_dist || d_off + margin < d_on);   // L98
    }
}

// -------------------------------------------------------------------------------------
// O13 IDM reactive sim agent (Fig. 2b): "follows the logged path ... but uses IDM
// to adjust the speed profile to avoid collisions and accelerate on free roads"; IDM = the
// intelligent driver model of ref. [51] (Treiber, Hennecke, Helbing 2000):
//     a = a_max [ 1 - (v / v0)^delta - (s* / s)^2 ],   s* = s0 + max(0, v T + v dv / (2 sqrt(a_max b)))
// with s the bumper-to-bumper gap to the lead object and dv = v - v_lead (no lead: last term 0).
// The paper gives no constants and no lead-finding rule; readings D37-D41:
//   D37 the constants are arguments (orc_idm_params; defaults declared in the Python wrapper);
//   D38 the path is the agent's on-route path (orc_paths), a polyline over index-consecutive valid
//       points; a position's path coordinate sigma is the arc length of its projection on the
//       nearest path segment (ties -> lower segment index);
//   D39 lead object: among the other agents valid at t, those whose projection on THIS agent's
//       path lies ahead (sigma_j > sigma_i) within a lateral distance of (W_i + W_j)/2; gap =
//       sigma_j - sigma_i - (L_i + L_j)/2; the smallest gap wins, ties -> lower agent index; lead
//       speed = |v_j|.  Projections and these decisions are taken in float32, operation for
//       operation as the kernel does (a floating-point value that decides an index);
//   D40 a is clamped to [-b_max, a_max], the gap to >= 0.1 m; v' = max(0, v + a dt); the agent
//       advances ds = (v + v') dt / 2 along its path: it lands on the first segment at or after its
//       own whose end lies beyond sigma_i + ds (linear interpolation), yaw' = that segment's
//       direction; past the end of the path it stays on the last point with its yaw;
//       velocity = v' (cos yaw', sin yaw'); length, width kept; valid' = 1;
//   D41 only agents with idm_valid != 0 that are valid at t and have a path segment are written
//       (row t+1); every other slot of row t+1 is left as it is (the caller's step fills it).
// -------------------------------------------------------------------------------------
struct orc_idm_params { float v0, T, s0, a_max, b, delta, b_max; };

struct PathProj { int k; float u, d2, sigma; };

// float32 projection of (qx, qy) on the segments (k, k+1) of agent a's path (D38)
static PathProj project_on_path(const orc_paths* pa, int b, int a, float qx, float qy) {
  const size_t o = ((size_t)b * pa->A + a) * pa->P;
  PathProj best{-1, 0.f, INFINITY, 0.f};
  for (int k = 0; k + 1 < pa->P; ++k) {
    if (!pa->valid[o + k] || !pa->valid[o + k + 1]) continue;
    const float ex = pa->x[o + k + 1] - pa->x[o + k], ey = pa->y[o + k + 1] - pa->y[o + k];
    const float wx = qx - pa->x[o + k], wy = qy - pa->y[o + k];
    const float ee = std::fmaf(ey, ey, ex * ex), dot = std::fmaf(wy, ey, wx * ex);
    float u = 0.f;
    if (ee > 0.f) u = std::fmin(std::fmax(dot / ee, 0.f), 1.f);
    const float rx = std::fmaf(-u, ex, wx), ry = std::fmaf(-u, ey, wy);
    const float d2 = std::fmaf(ry, ry, rx * rx);
    if (d2 < best.d2) { best.k = k; best.u = u; best.d2 = d2; }
  }
  if (best.k >= 0) best.sigma = std::fmaf(best.u, pa->arc_len[o + best.k + 1] - pa->arc_len[o + best.k], pa->arc_len[o + best.k]);
  return best;
}

void orc_idm_step(orc_traj* sim, int32_t t, const orc_paths* pa, const uint8_t* idm_valid, const orc_idm_params* prm, double dt,
                  float* accel_out, int32_t* lead_out) {
  const int B = sim->B, A = sim->A, P = pa->P;
#pragma omp parallel for schedule(static)
  for (int b = 0; b < B; ++b)
    for (int i = 0; i < A; ++i) {
      const size_t o = (size_t)b * A + i, r0 = row(sim, b, t) + i, r1 = row(sim, b, t + 1) + i;
      if (accel_out) accel_out[o] = 0.f;
      if (lead_out) lead_out[o] = -1;
      if (!idm_valid[o] || !sim->valid[r0]) continue;
      const PathProj self = project_on_path(pa, b, i, sim->x[r0], sim->y[r0]);
      if (self.k < 0) continue;                                                            // D41
      const size_t po = ((size_t)b * pa->A + i) * P;
      // ---- lead object (D39), float32 decisions ----
      int lead = -1;
      float gap = INFINITY;
      for (int j = 0; j < A; ++j) {
        const size_t rj = row(sim, b, t) + j;
        if (j == i || !sim->valid[rj]) continue;
        const PathProj pj = project_on_path(pa, b, i, sim->x[rj], sim->y[rj]);
        const float lat_max = 0.5f * (sim->width[r0] + sim->width[rj]);
        if (!(pj.sigma > self.sigma) || pj.d2 > lat_max * lat_max) continue;
        const float g = (pj.sigma - self.sigma) - 0.5f * (sim->length[r0] + sim->length[rj]);
        if (g < gap) { gap = g; lead = j; }
      }
      // ---- IDM acceleration (ref. [51]) ----
      const double vx = sim->vel_x[r0], vy = sim->vel_y[r0], v = std::sqrt(vx * vx + vy * vy);
      double acc = 1.0 - std::pow(v / prm->v0, (double)prm->delta);
      if (lead >= 0) {
        const size_t rl = row(sim, b, t) + lead;
        const double vl = std::sqrt((double)sim->vel_x[rl] * sim->vel_x[rl] + (double)sim->vel_y[rl] * sim->vel_y[rl]);
        const double sstar = prm->s0 + std::max(0.0, v * prm->T + v * (v - vl) / (2.0 * std::sqrt((double)prm->a_max * prm->b)));
        const double sgap = std::max((double)gap, 0.1);
        acc -= (sstar / sgap) * (sstar / sgap);
      }
      acc *= prm->a_max;
      acc = std::min(std::max(acc, -(double)prm->b_max), (double)prm->a_max);              // D40
      const double v1 = std::max(0.0, v + acc * dt);
      const double target = (double)self.sigma + 0.5 * (v + v1) * dt;
      // ---- advance along the path (D40) ----
      int ks = -1;
      for (int k = self.k; k + 1 < P; ++k)
        if (pa->valid[po + k] && pa->valid[po + k + 1] && (double)pa->arc_len[po + k + 1] > target) { ks = k; break; }
      double xn, yn, yawn;
      if (ks >= 0) {
        const double ex = (double)pa->x[po + ks + 1] - pa->x[po + ks], ey = (double)pa->y[po + ks + 1] - pa->y[po + ks];
        const double len = (double)pa->arc_len[po + ks + 1] - pa->arc_len[po + ks];
        const double u = std::min(std::max((target - pa->arc_len[po + ks]) / len, 0.0), 1.0);
        xn = pa->x[po + ks] + u * ex; yn = pa->y[po + ks] + u * ey; yawn = std::atan2(ey, ex);
      } else {                                                                             // past the end: the last path point
        int kl = self.k + 1;
        for (int k = self.k + 1; k < P; ++k) if (pa->valid[po + k] && pa->valid[po + k - 1]) kl = k; else break;
        xn = pa->x[po + kl]; yn = pa->y[po + kl]; yawn = sim->yaw[r0];
      }
      sim->x[r1] = (float)xn; sim->y[r1] = (float)yn; sim->yaw[r1] = (float)yawn;
      sim->vel_x[r1] = (float)(v1 * std::cos(yawn)); sim->vel_y[r1] = (float)(v1 * std::sin(yawn));
      sim->length[r1] = sim->length[r0]; sim->width[r1] = sim->width[r0]; sim->valid[r1] = 1;
      if (accel_out) accel_out[o] = (float)acc;
      if (lead_out) lead_out[o] = lead;
    }
}

// -------------------------------------------------------------------------------------
// O14 backward pass of the dynamics ("the entire simulation can be assembled within a
// single ... computation graph" / differentiable simulation): the vector-Jacobian
// product of O1 / O2, chained in reverse over the rows of a rollout.  Plain reverse-mode
// differentiation of Eq. 2 (L339-L350) and Eq. 1 (L324-L333) written out term by term, in double,
// evaluated on the STORED float32 rows (state at row t0+k, actions of step k).  Readings (DESIGN D43):
//   * a playback slot (use_dyn = action_valid && sim.valid[t0+k] false, D8) takes its successor from
//     the log: zero gradient to the state and to the action;
//   * clipping (D7): d clip(a)/da = 1 for |a| <= limit, 0 beyond it;
//   * v = sqrt(vx^2 + vy^2): dv/dvx = vx / v, and 0 at v = 0;
//   * Eq. 1's v' = (x' - x)/dt differentiates as written (the float32 rounding of x', D28, is the
//     identity for the derivative): for the delta models v' does not depend on x.
// g_rows [B][n_steps][5][A]: cotangents of the loss w.r.t. (x, y, yaw, vel_x, vel_y) of rows
// t0+1 .. t0+n_steps.  Outputs: g_actions [B][n_steps][C][A], g_state0 [B][5][A] (w.r.t. row t0).
// -------------------------------------------------------------------------------------
void orc_rollout_vjp(const orc_traj* sim, int32_t t0, int32_t n_steps, int32_t dynamics, double dt, double max_accel,
                     double max_curvature, const float* actions, const uint8_t* action_valid, const float* g_rows,
                     float* g_actions, float* g_state0) {
  const int B = sim->B, A = sim->A;
  const int C = dynamics == ORC_DYN_BICYCLE ? 2 : 3;
#pragma omp parallel for schedule(static)
  for (int b = 0; b < B; ++b)
    for (int a = 0; a < A; ++a) {
      double gx = 0, gy = 0, gth = 0, gvx = 0, gvy = 0;            // cotangent of row t0+k+1, carried backwards
      for (int k = n_steps - 1; k >= 0; --k) {
        const size_t gr = (((size_t)b * n_steps + k) * 5) * A + a;
        gx += g_rows[gr]; gy += g_rows[gr + A]; gth += g_rows[gr + 2 * (size_t)A];
        gvx += g_rows[gr + 3 * (size_t)A]; gvy += g_rows[gr + 4 * (size_t)A];
        const size_t r0 = row(sim, b, t0 + k) + a;
        const size_t oa = (((size_t)b * n_steps + k) * C) * A + a;
        const bool use_dyn = action_valid[((size_t)b * n_steps + k) * A + a] != 0 && sim->valid[r0] != 0;
        for (int c = 0; c < C; ++c) g_actions[oa + (size_t)c * A] = 0.f;
        if (!use_dyn) { gx = gy = gth = gvx = gvy = 0; continue; }  // the successor came from the log
        const double th = sim->yaw[r0], vx = sim->vel_x[r0], vy = sim->vel_y[r0];
        double nx_, ny_, nth, nvx, nvy;                             // cotangent of row t0+k
        if (dynamics == ORC_DYN_BICYCLE) {
          double acc = actions[oa], kappa = actions[oa + A];
          double da = 1.0, dk = 1.0;
          if (max_accel > 0) { if (std::fabs(acc) > max_accel) da = 0.0; acc = std::min(std::max(acc, -max_accel), max_accel); }
          if (max_curvature > 0) { if (std::fabs(kappa) > max_curvature) dk = 0.0; kappa = std::min(std::max(kappa, -max_curvature), max_curvature); }
          const double v = std::sqrt(vx * vx + vy * vy);
          const double thn = th + kappa * (v * dt + 0.5 * acc * dt * dt);   // L343
          const double vn = v + acc * dt;                                    // L345
          const double c0 = std::cos(th), s0 = std::sin(th), c1 = std::cos(thn), s1 = std::sin(thn);
          // vx' = vn cos(thn), vy' = vn sin(thn)                           (L347, L349)
          const double gvn = gvx * c1 + gvy * s1;
          const double gthn = gth + vn * (-gvx * s1 + gvy * c1);
          // thn = th + kappa (v dt + a dt^2/2)
          const double gv = gvn + gthn * kappa * dt;
          const double gk = gthn * (v * dt + 0.5 * acc * dt * dt);
          // x' = x + vx dt + a cos(th) dt^2/2, y' = y + vy dt + a sin(th) dt^2/2   (L339, L341)
          const double ga = gvn * dt + gthn * kappa * 0.5 * dt * dt + 0.5 * dt * dt * (gx * c0 + gy * s0);
          nth = gthn + 0.5 * acc * dt * dt * (-gx * s0 + gy * c0);
          nx_ = gx; ny_ = gy;
          const double ux = v > 0 ? vx / v : 0.0, uy = v > 0 ? vy / v : 0.0;
          nvx = gx * dt + gv * ux; nvy = gy * dt + gv * uy;
          g_actions[oa] = (float)(ga * da); g_actions[oa + A] = (float)(gk * dk);
        } else {
          const double dx = actions[oa], dy = actions[oa + A];
          const bool glob = dynamics == ORC_DYN_DELTA_GLOBAL;
          const double c = glob ? 1.0 : std::cos(th), s = glob ? 0.0 : std::sin(th);
          // x' = x + c dx - s dy, y' = y + s dx + c dy, th' = th + dyaw, vx' = (x' - x)/dt, vy' = (y' - y)/dt
          const double hx = gx + gvx / dt, hy = gy + gvy / dt;      // cotangents of the world-frame delta
          g_actions[oa] = (float)(hx * c + hy * s);
          g_actions[oa + A] = (float)(-hx * s + hy * c);
          g_actions[oa + 2 * (size_t)A] = (float)gth;
          nx_ = gx; ny_ = gy;
          nth = gth + (glob ? 0.0 : hx * (-s * dx - c * dy) + hy * (c * dx - s * dy));
          nvx = 0.0; nvy = 0.0;
        }
        gx = nx_; gy = ny_; gth = nth; gvx = nvx; gvy = nvy;
      }
      const size_t o = ((size_t)b * 5) * A + a;
      g_state0[o] = (float)gx; g_state0[o + A] = (float)gy; g_state0[o + 2 * (size_t)A] = (float)gth;
      g_state0[o + 3 * (size_t)A] = (float)gvx; g_state0[o + 4 * (size_t)A] = (float)gvy;
    }
}

// -------------------------------------------------------------------------------------
// O15 discretised action spaces ("For discrete action spaces, the inverse is computed by
// discretizing the continuous inverse"; the Bicycle-Discrete / Delta-Discrete spaces of L373).  The
// paper prints no grids, so they are arguments (DESIGN D42): channel c has n[c] >= 1 values
// lo[c] + i (hi[c] - lo[c]) / (n[c] - 1), i = 0 .. n[c]-1 (n = 1: the single value lo).  A continuous
// value maps to the NEAREST grid value, ties to the even bin, beyond the range to the end bin.  The
// bin decision is taken in float32 (the kernel's precision: a floating-point value that decides an
// integer): i = clamp(rint((v - lo) * inv_step), 0, n-1) with inv_step = (n-1)/(hi-lo) rounded to
// float32 and every operation rounded to float32.  The joint index is row-major over the channels,
// index = (i_0 n_1 + i_1) n_2 + i_2.  The de-quantised value is lo + i step in double, rounded once.
// action [N][C][A] -> index [N][A] (N = B n_steps rows), dequant [N][C][A] (may be NULL).
// -------------------------------------------------------------------------------------
struct orc_action_grid { int32_t n[3]; float lo[3], hi[3]; };

void orc_discretize_actions(const orc_action_grid* g, int32_t C, int64_t N, int32_t A, const float* action, const uint8_t* valid,
                            int32_t* index, float* dequant) {
  for (int64_t r = 0; r < N; ++r)
    for (int a = 0; a < A; ++a) {
      int32_t idx = 0;
      const bool v = valid == nullptr || valid[r * A + a] != 0;
      for (int c = 0; c < C; ++c) {
        const size_t o = ((size_t)r * C + c) * A + a;
        int i = 0;
        if (v && g->n[c] > 1) {
          const float inv_step = (float)(g->n[c] - 1) / (g->hi[c] - g->lo[c]);
          const float q = std::nearbyintf((action[o] - g->lo[c]) * inv_step);        // round half to even, float32
          i = q <= 0.f ? 0 : q >= (float)(g->n[c] - 1) ? g->n[c] - 1 : (int)q;       // NaN -> bin 0
          if (!(q == q)) i = 0;
        }
        idx = idx * g->n[c] + i;
        if (dequant) {
          const double step = g->n[c] > 1 ? ((double)g->hi[c] - (double)g->lo[c]) / (double)(g->n[c] - 1) : 0.0;
          dequant[o] = v ? (float)((double)g->lo[c] + (double)i * step) : 0.f;
        }
      }
      index[r * A + a] = v ? idx : -1;
    }
}

// joint index -> continuous action (the de-quantised grid value; index < 0 -> 0; D45: an index that is not
// a bin of the grid, index >= n_0 n_1 .. n_{C-1}, is no action either -> 0)
void orc_actions_from_index(const orc_action_grid* g, int32_t C, int64_t N, int32_t A, const int32_t* index, float* action) {
  int64_t total = 1;
  for (int c = 0; c < C; ++c) total *= g->n[c];
  for (int64_t r = 0; r < N; ++r)
    for (int a = 0; a < A; ++a) {
      int32_t idx = index[r * A + a];
      if ((int64_t)idx >= total) idx = -1;
      for (int c = C - 1; c >= 0; --c) {
        const size_t o = ((size_t)r * C + c) * A + a;
        if (idx < 0) { action[o] = 0.f; continue; }
        const int i = idx % g->n[c];
        idx /= g->n[c];
        const double step = g->n[c] > 1 ? ((double)g->hi[c] - (double)g->lo[c]) / (double)(g->n[c] - 1) : 0.0;
        action[o] = (float)((double)g->lo[c] + (double)i * step);
      }
    }
}

int32_t orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
