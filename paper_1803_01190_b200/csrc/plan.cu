// plan.cu -- host-side launch plan of one gravity solve (no device code).
//
// The all-pairs sweep of eq. (1) is cut into (i-block, j-split) work units.  The paper's Kepler GPUs
// had 13-15 SMs, so "one thread per i-particle" filled them at any N of interest; a B200 has 148 SMs
// and N = 2^20 bodies in 1792-body i-blocks are only 3.96 waves.  The plan therefore picks the shape class (large /
// mid / small, ppgrav_internal.h; by calibrated size thresholds) and the split factor S that minimises
//     waves x (tiles per split + fixed overhead) x tile cost  +  weight x S x bodies
// so that the last wave is nearly full.  The class thresholds and the weight are calibrated on the B200 with the
// throughput-vs-N sweep of `bench.py --sweep-n` (raw data profiles/r2_sweep_n.json).
#include <algorithm>
#include <cmath>

#include "ppgrav_internal.h"

namespace ppgrav {

namespace {

// Which shape class serves a solve of i_count i-bodies against N j-bodies: calibrated on the B200 with
// `bench.py --sweep-n` (profiles/r2_sweep_n.json), where every class was pinned in turn at
// N = 2^11 .. 2^21.  The fastest class (whole pp_forces call, force only) was
//   FP32: small up to 2^13, mid at 2^14, large from 2^15;     FP64: small up to 2^14, large from 2^15
// (the FP64 mid class never beat both neighbours; it stays reachable through PP_CFG_SHAPE).  A range solve is placed by
// the geometric mean of its two sides.
int calibrated_class(int precision, int64_t N, int64_t i_count) {
    const double n_eff = std::sqrt((double)N * (double)i_count);
    if (precision == PP_F64) return n_eff < 24000.0 ? CLS_SMALL : CLS_LARGE;
    return n_eff < 12000.0 ? CLS_SMALL : n_eff < 24000.0 ? CLS_MID : CLS_LARGE;
}

// relative cost of a tile in a class (large = 1), used only to weigh a class's sweep against its partial-sum traffic
// when S is chosen: the values S was calibrated with in round 1
constexpr double kClassWeight[2][kNumClasses] = {
    /* PP_F32 */ {1.0, 0.90, 0.45},
    /* PP_F64 */ {1.0, 0.93, 0.80},
};

int64_t round_up(int64_t a, int64_t b) { return (a + b - 1) / b * b; }

// weight of one split-j partial sum of one body (written by the sweep, read by the finalize pass), in pair
// interactions of one SM.  The bandwidth cost alone is ~0.1; the weight is larger so that a bigger S is only taken when
// it fills the last wave noticeably better.
constexpr double kFinalizeCost = 16.0;
// the same for the symmetric sweep, whose tile costs 29 us against ~1.4 us for writing and re-reading one more
// partial sum per body at N = 2^17: a small weight, so that S = 8-9 fills the 148 SMs at N = 2^17 .. 2^18, where
// 64-128 blocks alone leave a seventh of them idle
constexpr double kSymFinalizeCost = 2.0;

}  // namespace

Plan make_plan(int64_t N, int precision, int mode, int sm_count, int64_t forced_split, int forced_cls, int64_t i_begin,
               int64_t i_count) {
    if (i_count < 0) i_count = N - i_begin;
    Plan best{};
    double best_cost = -1.0;
    const int pi = precision == PP_F64 ? 1 : 0;
    const size_t elem = precision == PP_F64 ? 32 : 16;
    const int cls = (forced_cls >= 0 && forced_cls < kNumClasses) ? forced_cls : calibrated_class(precision, N, i_count);
    for (int c = cls; c <= cls; ++c) {
        const KernelShape& d = kShapes[pi][c][mode];
        Plan p{};
        p.cls = c;
        p.mode = mode;
        p.threads = d.threads;
        p.ipt = d.ipt;
        p.i_per_cta = d.threads * d.ipt;
        p.tile_j = d.tile_j;
        p.stages = d.stages;
        p.ctas_per_sm = d.ctas_per_sm;
        p.sm_count = sm_count;
        p.i_begin = i_begin;
        p.i_count = i_count;
        p.n_iblocks = (int)((i_count + p.i_per_cta - 1) / p.i_per_cta);
        p.part_stride = (int64_t)p.n_iblocks * p.i_per_cta;
        // the packed array must cover the last launched i-block (which may reach past N) and the last j-tile
        p.n_pad = round_up(std::max(N, i_begin + p.part_stride), p.tile_j);
        p.n_tiles = (int)((N + p.tile_j - 1) / p.tile_j);
        const int64_t resident = (int64_t)sm_count * d.ctas_per_sm;
        // partial sums: S x part_stride x {16,32} bytes, kept under 1 GiB
        int64_t s_max = std::min<int64_t>(std::min<int64_t>(p.n_tiles, 64),
                                          std::max<int64_t>(1, (int64_t)((1ull << 30) / (p.part_stride * elem))));
        int64_t s_lo = 1, s_hi = s_max;
        if (forced_split >= 1) s_lo = s_hi = std::min<int64_t>(forced_split, p.n_tiles);
        const double tile_cost = (double)p.i_per_cta * p.tile_j * d.ctas_per_sm / kClassWeight[pi][c];
        for (int64_t S = s_lo; S <= s_hi; ++S) {
            const int64_t units = (int64_t)p.n_iblocks * S;
            const int64_t waves = (units + resident - 1) / resident;
            const int64_t tps = (p.n_tiles + S - 1) / S;
            // 2 tile-times of fixed cost per unit (pipeline fill, epilogue), plus the finalize pass over S partials
            const double cost = (double)waves * ((double)tps + 2.0) * tile_cost + kFinalizeCost * (double)S * (double)p.part_stride;
            if (best_cost < 0.0 || cost < best_cost * (1.0 - 1e-9)) {
                best_cost = cost;
                best = p;
                best.split = (int)S;
            }
        }
    }
    return best;
}

Plan make_sym_plan(int64_t N, int precision, int mode, int sm_count, int64_t forced_split, size_t rows_cap_bytes,
                   size_t* jbytes, size_t* abytes, int fine_tiles) {
    const bool fine = fine_tiles < 0 ? N < kSymFineBelow : fine_tiles != 0;
    const KernelShape& d = precision == PP_F64 ? (fine ? kShapeF64SymFine : kShapeF64Sym)
                                               : (fine ? kShapeF32SymFine : kShapeF32Sym);
    const size_t elem = precision == PP_F64 ? 32 : 16;
    Plan p{};
    p.cls = CLS_LARGE;
    p.mode = mode;
    p.threads = d.threads;
    p.ipt = d.ipt;
    p.i_per_cta = d.threads * d.ipt;
    p.tile_j = d.tile_j;
    p.stages = d.stages;
    p.ctas_per_sm = d.ctas_per_sm;
    p.sm_count = sm_count;
    p.i_begin = 0;
    p.i_count = N;
    p.n_iblocks = (int)((N + p.i_per_cta - 1) / p.i_per_cta);
    p.part_stride = (int64_t)p.n_iblocks * p.i_per_cta;
    p.n_pad = p.part_stride;                      // whole blocks: the cyclic partner ranges wrap over the padding
    p.n_tiles = (int)(p.part_stride / p.tile_j);  // every tile of every block is swept (padding is massless)
    p.sym = 1;
    p.sym_h = (p.n_iblocks - 1) / 2;
    // split-j over the partner tiles of a block: fill the last wave, as make_plan does
    const int tpb = p.i_per_cta / p.tile_j;
    const int64_t ptiles = (int64_t)p.sym_h * tpb;
    int64_t s_lo = 1, s_hi = std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(ptiles + tpb, 64),
                                                                     (int64_t)((1ull << 30) / (p.part_stride * elem))));
    if (forced_split >= 1) s_lo = s_hi = std::max<int64_t>(1, std::min<int64_t>(forced_split, ptiles + tpb));
    double best = -1.0;
    p.split = 1;
    for (int64_t S = s_lo; S <= s_hi; ++S) {
        const int64_t units = (int64_t)p.n_iblocks * S;
        const int64_t waves = (units + sm_count - 1) / sm_count;
        // per unit: its share of the block's tiles (the one-sided ones of the own and, for an even block count, the
        // opposite block, plus the partner tiles) + 2 tile-times of fill and epilogue
        const double n_ns = (double)tpb * ((p.n_iblocks > 1 && p.n_iblocks % 2 == 0) ? 2.0 : 1.0);
        const double per_unit = std::ceil(((double)ptiles + n_ns) / (double)S) + 2.0;
        const double cost = (double)waves * per_unit * p.i_per_cta * p.tile_j +
                            kSymFinalizeCost * (double)S * (double)p.part_stride;
        if (best < 0.0 || cost < best * (1.0 - 1e-9)) { best = cost; p.split = (int)S; }
    }
    // bands: as many partner offsets per band as rows_cap_bytes holds
    const size_t row_bytes = (size_t)p.part_stride * elem;
    p.sym_rows = (int)std::max<size_t>(1, std::min<size_t>((size_t)std::max(p.sym_h, 1), rows_cap_bytes / row_bytes));
    p.sym_bands = std::max(1, (p.sym_h + p.sym_rows - 1) / p.sym_rows);
    // a banded solve (N > 2^21: thousands of blocks per band) needs no split-j
    if (p.sym_bands > 1 && forced_split < 1) p.split = 1;
    if (jbytes) *jbytes = std::max<size_t>((size_t)std::min(p.sym_rows, std::max(p.sym_h, 1)) * row_bytes, 16);
    if (abytes) *abytes = p.sym_bands > 1 ? 2 * row_bytes : 0;
    return p;
}

}  // namespace ppgrav
