// Experiment switches.  The DEFAULT build has none: debug_env() returns compile-time constants and the library reads
// no environment variable.  Only a build with -DSHARQ_EXPERIMENTS (never shipped; used for sweeps and ablations)
// reads the SHARQ_DEBUG_* variables below, once per process.
#pragma once
#include <cstdlib>

namespace sharq {

struct DebugEnv {
  int no_pdl;          // SHARQ_DEBUG_NO_PDL: launch without programmatic dependent launch
  int grid;            // SHARQ_DEBUG_GRID: CTAs of the persistent 1-CTA GEMM (0 = default)
  int pair_clusters;   // SHARQ_DEBUG_PAIR_CLUSTERS: cap on the clusters of the pair GEMM (0 = default)
  int no_pair;         // SHARQ_DEBUG_NO_PAIR=1: never use the pair GEMM
  int force_pair;      // SHARQ_DEBUG_FORCE_PAIR=1: pair GEMM whenever T > 128
  int pair_bn;         // SHARQ_DEBUG_PAIR_BN: force the pair tile width (192 / 256; 0 = cost model)
  int no_mc;           // SHARQ_DEBUG_NO_MC: grouped GEMM without multicast clusters
  int wide_t;          // SHARQ_DEBUG_WIDE_T: largest T for 128 x 256 tiles (default 128)
  int no_wide;         // SHARQ_DEBUG_NO_WIDE: never use 128 x 256 tiles
  int row_per_sm;      // SHARQ_DEBUG_ROW_PER_SM: prepare grid = this many CTAs per SM (0 = default)
  int old_prepare;     // SHARQ_DEBUG_OLD_PREPARE: warp-per-row prepare kernel for every K
  int pair_gm;         // SHARQ_DEBUG_PAIR_GM: supertile height of the pair GEMM in 256-row blocks (0 = by L2 footprint)
  int skip_prep;       // SHARQ_DEBUG_SKIP_PREP: fused decode launch without its in-kernel prepare (timing experiment)
  int prep_chunk_rows; // SHARQ_DEBUG_PREP_CHUNK_ROWS: rows per launch of the row-per-CTA prepare kernel (tests; 0 = 2^31 / width)
};

#ifndef SHARQ_EXPERIMENTS
constexpr DebugEnv kNoDebug{0, 0, 0, 0, 0, 0, 0, 128, 0, 0, 0, 0, 0, 0};
inline constexpr const DebugEnv& debug_env() { return kNoDebug; }
#else
inline const DebugEnv& debug_env() {
  static const DebugEnv e = [] {
    auto num = [](const char* name, int dflt) {
      const char* v = std::getenv(name);
      return v ? std::atoi(v) : dflt;
    };
    auto flag = [](const char* name) { return std::getenv(name) ? 1 : 0; };
    DebugEnv d;
    d.no_pdl = flag("SHARQ_DEBUG_NO_PDL");
    d.grid = num("SHARQ_DEBUG_GRID", 0);
    d.pair_clusters = num("SHARQ_DEBUG_PAIR_CLUSTERS", 0);
    d.no_pair = num("SHARQ_DEBUG_NO_PAIR", 0) == 1;
    d.force_pair = num("SHARQ_DEBUG_FORCE_PAIR", 0) == 1;
    d.pair_bn = num("SHARQ_DEBUG_PAIR_BN", 0);
    d.no_mc = flag("SHARQ_DEBUG_NO_MC");
    d.wide_t = num("SHARQ_DEBUG_WIDE_T", 128);
    d.no_wide = flag("SHARQ_DEBUG_NO_WIDE");
    d.row_per_sm = num("SHARQ_DEBUG_ROW_PER_SM", 0);
    d.old_prepare = flag("SHARQ_DEBUG_OLD_PREPARE");
    d.pair_gm = num("SHARQ_DEBUG_PAIR_GM", 0);
    d.skip_prep = flag("SHARQ_DEBUG_SKIP_PREP");
    d.prep_chunk_rows = num("SHARQ_DEBUG_PREP_CHUNK_ROWS", 0);
    return d;
  }();
  return e;
}
#endif

}  // namespace sharq
