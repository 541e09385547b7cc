// plan.cu -- host-only planning helpers: the workspace layout, the module-level roofline fit and the
// B_moe choice (include/bg_moe.h; §5.1, §5.4).  No device code.
#include "kernels.h"

#include <cmath>
#include <limits>

namespace bg {

WsLayout ws_layout(const bg_moe_config& c, int64_t max_tokens, int num_sms) {
  const int64_t Tm = max_tokens > 0 ? max_tokens : 1;
  const int64_t Rm = Tm * c.k;
  const int64_t ntile = route_num_tiles(static_cast<int>(Tm));
  int64_t off = 0;
  auto carve = [&](int64_t bytes) {
    const int64_t o = off;
    off = (off + bytes + 1023) / 1024 * 1024;
    return o;
  };
  (void)num_sms;
  WsLayout L;
  L.logits = carve(Tm * c.E * 4);
  L.idx = carve(Rm * 4);
  L.w = carve(Rm * 4);
  L.pieces = carve(3LL * c.d * ((c.E + 15) & ~15) * 2);
  L.counts = carve(c.E * 4);
  L.offsets = carve((c.E + 1) * 4);
  L.tc = carve(ntile * c.E * 4);     // per-tile expert histograms
  L.tb = carve(ntile * c.E * 4);     // per-tile base rows
  L.tr = carve(Rm * 4);              // tile-local ranks
  L.rs = carve(Rm * 4);
  L.ip = carve(Rm * 4);
  L.wp = carve(Rm * 4);
  L.x = carve(Rm * c.d * 2);
  L.h = carve(Rm * c.f * 2);
  L.y = carve(Rm * c.d * 2);
  L.hd = carve(2 * Tm * c.d * 2);    // host entry point: two staging slots each way
  L.od = carve(2 * Tm * c.d * 2);
  // segment table (at most max_tokens segments), ONE slab so that one copy can fill it:
  // hidden[Tm] pointers | out[Tm] pointers | start[Tm + 1] ints
  L.seg_hidden = carve(16 * Tm + 4 * (Tm + 1));
  L.seg_out = L.seg_hidden + 8 * Tm;
  L.seg_start = L.seg_hidden + 16 * Tm;
  L.tile_counters = carve(64);       // [0..7] GEMM ticket counters, [8] router tiles-done counter
  L.total = off;
  return L;
}

namespace {

bool config_ok(const bg_moe_config* c) {
  return c != nullptr && c->d >= 64 && c->f >= 64 && c->d % 8 == 0 && c->f % 8 == 0 && c->E >= 1 && c->E <= 256 &&
         c->k >= 1 && c->k <= c->E && c->k <= 8;
}

double model_ms(const bg_moe_fit& f, double T) { return std::fmax(f.t_floor_ms, f.t0_ms + f.ms_per_token * T); }

}  // namespace
}  // namespace bg

extern "C" {

int bg_moe_fit_roofline(const int32_t* tokens, const double* ms, int32_t n, bg_moe_fit* out) {
  if (tokens == nullptr || ms == nullptr || out == nullptr || n < 3) return BG_ERR_INVALID_ARG;
  for (int i = 0; i < n; ++i) {
    if (!(ms[i] > 0.0) || tokens[i] < 0) return BG_ERR_INVALID_ARG;
    if (i > 0 && tokens[i] <= tokens[i - 1]) return BG_ERR_INVALID_ARG;
  }
  double best = std::numeric_limits<double>::infinity();
  bg_moe_fit best_fit = {};
  for (int j = 1; j <= n - 2; ++j) {
    double flat = 0.0;
    for (int i = 0; i < j; ++i) flat += ms[i];
    flat /= j;
    // ordinary least squares on the points j .. n-1
    const int m = n - j;
    double sx = 0, sy = 0, sxx = 0, sxy = 0;
    for (int i = j; i < n; ++i) {
      const double x = tokens[i], y = ms[i];
      sx += x; sy += y; sxx += x * x; sxy += x * y;
    }
    const double den = m * sxx - sx * sx;
    if (!(den > 0.0)) continue;
    const double slope = (m * sxy - sx * sy) / den;
    const double icpt = (sy - slope * sx) / m;
    if (!(slope > 0.0)) continue;
    bg_moe_fit f;
    f.t_floor_ms = flat;
    f.t0_ms = icpt;
    f.ms_per_token = slope;
    f.ridge_tokens = (flat - icpt) / slope;
    double sse = 0.0;
    for (int i = 0; i < n; ++i) {
      const double r = (bg::model_ms(f, tokens[i]) - ms[i]) / ms[i];
      sse += r * r;
    }
    f.rms_rel_err = std::sqrt(sse / n);
    if (sse < best) {
      best = sse;
      best_fit = f;
    }
  }
  if (!std::isfinite(best)) return BG_ERR_INVALID_ARG;
  *out = best_fit;
  return BG_OK;
}

int bg_moe_workspace_bytes_for(const bg_moe_config* cfg, int32_t tokens, int64_t* bytes_out) {
  if (!bg::config_ok(cfg) || tokens < 0 || bytes_out == nullptr) return BG_ERR_INVALID_ARG;
  if (static_cast<int64_t>(tokens) * cfg->k > 0x7fffffffLL) return BG_ERR_INVALID_ARG;
  *bytes_out = bg::ws_layout(*cfg, tokens, 148).total;
  return BG_OK;
}

int bg_moe_choose_tokens(const bg_moe_config* cfg, const bg_moe_fit* fit, double target_util,
                         int64_t memory_budget_bytes, int32_t granularity, int32_t* tokens_out,
                         int32_t* reached_out) {
  if (!bg::config_ok(cfg) || fit == nullptr || tokens_out == nullptr || granularity < 1) return BG_ERR_INVALID_ARG;
  if (!(target_util > 0.0 && target_util < 1.0) || !(fit->ms_per_token > 0.0) || !(fit->t_floor_ms > 0.0))
    return BG_ERR_INVALID_ARG;
  // largest multiple of `granularity` whose workspace fits: the layout grows monotonically with tokens
  const int64_t cap_tokens = 0x7fffffffLL / cfg->k / granularity * granularity;
  auto fits = [&](int64_t T) { return bg::ws_layout(*cfg, T, 148).total <= memory_budget_bytes; };
  if (!fits(granularity)) return BG_ERR_NOMEM;
  int64_t lo = 1, hi = cap_tokens / granularity;       // in units of granularity; fits(lo) holds
  while (lo < hi) {
    const int64_t mid = lo + (hi - lo + 1) / 2;
    if (fits(mid * granularity)) lo = mid; else hi = mid - 1;
  }
  const int64_t t_mem = lo * granularity;
  // smallest multiple of `granularity` with u(T) = min(1, s T / max(floor, t0 + s T)) >= target.  u is
  // non-decreasing in T: rising on the flat part, and on the line either rising towards 1 (t0 >= 0)
  // or clipped at 1 (t0 < 0), so a binary search finds the first T that reaches the target.
  auto util = [&](int64_t T) {
    return std::fmin(1.0, fit->ms_per_token * T / bg::model_ms(*fit, static_cast<double>(T)));
  };
  int64_t t_util = -1;
  if (util(t_mem) >= target_util) {
    int64_t a = 1, b = t_mem / granularity;            // util(b * g) >= target
    while (a < b) {
      const int64_t mid = a + (b - a) / 2;
      if (util(mid * granularity) >= target_util) b = mid; else a = mid + 1;
    }
    t_util = a * granularity;
  }
  const bool reached = t_util > 0;
  *tokens_out = static_cast<int32_t>(reached ? t_util : t_mem);
  if (reached_out != nullptr) *reached_out = reached ? 1 : 0;
  return BG_OK;
}

}  // extern "C"
