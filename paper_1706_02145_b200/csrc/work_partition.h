// work_partition.h -- how the N x N pair grid of one matvec is cut into work for the coupling kernel (host side).
//
// Receivers are grouped into receiver blocks of `bs` <= kBlock consecutive spheres (one thread each); the emitter sum
// of a block is walked in tiles of `etile` emitters.  A SEGMENT is (receiver block r, emitters [e_begin, e_end), slot):
// the CTA that owns it accumulates those emitters into fresh accumulators and stores them in partial-sum slot `slot`;
// finalize_kernel adds the slots of a block in slot order, which is fixed by this table alone, so results are
// reproducible bit for bit and do not depend on which CTAs ran or on a restriction to a slice of receiver rows.
//
//   guided (default): the rblocks x tiles grid is flattened, receiver block major, and cut into LEVELS of runs: the
//       first level covers half of the tiles in n_res equal runs (n_res = SMs x resident CTAs, one wave), the next a
//       quarter, ... the last two a 2^-(levels-1) share each.  The hardware dispatches CTAs in launch order as slots
//       free up, so the short runs at the end even out what the long ones leave uneven -- and they leave a lot: of two
//       CTAs resident on an SM the warp scheduler favours one almost exclusively (measured: it finishes after 58 % of the
//       pair's time, profiles/r02_cta_trace.md), and a CTA left alone on an SM reaches only 92 % of the pipe throughput
//       of two.  One level (a single wave of equal runs) is 5.5 % slower than many waves for that reason; at N = 1e5
//       six levels take 357.25 ms, ten (the default) 355.90 ms and more change nothing.  The halving stops once a run would
//       be shorter than CELES_MIN_RUN_TILES = 16 emitter tiles: at N = 1e4 that gives three levels with tiles of 32, measured
//       best there (lmax 4: 7.440 ms against 7.476 with five and 7.719 with one; the 965 partial sums then stay in L2 --
//       0.55 MB of DRAM writes per launch against 22.9 MB with five levels -- and finalize_kernel takes 20 us instead of 44),
//       and five levels with the tiles of 8 of lmax = 5, measured slightly better for that kernel (18.06 ms against 18.2 with three).
//       At most n_res * levels + rblocks partial sums, instead of 56 per receiver block at N = 1e4 with fixed splits.
//   fixed splits (celes_options.emitter_splits = S > 0): every block's emitters are cut into S equal chunks, one CTA
//       each, grid = rblocks x S CTAs in as many waves as that takes.
#pragma once
#include <algorithm>
#include <vector>

#ifndef CELES_MIN_RUN_TILES
#define CELES_MIN_RUN_TILES 16    // shortest run the halving may produce, in emitter tiles (note above)
#endif

namespace celes {

struct Segment {
    int rblock;    // receiver block
    int e_begin;   // first emitter
    int e_end;     // one past the last emitter
    int slot;      // partial-sum slot written: ypart[slot][thread][q]
};

struct WorkPartition {
    int bs = 0, rblocks = 0, n_cta = 0;
    std::vector<Segment> seg;          // ordered by CTA (launch order); within a CTA by (rblock, e_begin)
    std::vector<int> cta_begin;        // [n_cta + 1] first segment of each CTA
    std::vector<int> slot_begin;       // [rblocks + 1] first slot of each receiver block: the slots of a block are
                                       // contiguous and ordered by e_begin, whichever CTAs produce them
};

inline WorkPartition build_partition(int N, int kblock, int etile, int n_res, int levels, int fixed_splits) {
    WorkPartition p;
    p.rblocks = (N + kblock - 1) / kblock;
    p.bs = (N + p.rblocks - 1) / p.rblocks;                 // receivers spread evenly: no nearly empty last block
    p.rblocks = (N + p.bs - 1) / p.bs;
    const long long tiles = (N + etile - 1) / etile;        // emitter tiles per receiver block
    const long long total = tiles * p.rblocks;
    const long long min_run_tiles = CELES_MIN_RUN_TILES;
    // runs of consecutive tiles of the flattened grid, one per CTA, in launch order
    std::vector<std::pair<long long, long long>> runs;
    if (fixed_splits > 0) {
        const int S = (int)std::min<long long>(fixed_splits, tiles);
        const long long per = (tiles + S - 1) / S;
        for (int r = 0; r < p.rblocks; ++r)
            for (long long t0 = 0; t0 < tiles; t0 += per) runs.push_back({r * tiles + t0, r * tiles + std::min(tiles, t0 + per)});
    } else {
        long long done = 0;
        for (int lev = 0; lev < std::max(1, levels) && done < total; ++lev) {
            const bool last = lev + 1 >= std::max(1, levels);
            long long share = last ? total - done : (total - done) / 2;
            if (share < min_run_tiles * n_res) share = total - done;       // shorter runs would not pay: stop halving
            const long long n = std::max<long long>(1, std::min<long long>(n_res, share));
            for (long long c = 0; c < n; ++c) {
                const long long a = done + share * c / n, b = done + share * (c + 1) / n;
                if (b > a) runs.push_back({a, b});
            }
            done += share;
        }
    }
    p.n_cta = (int)runs.size();
    std::vector<int> nseg_of_block(p.rblocks, 0);
    for (const auto& run : runs) {
        p.cta_begin.push_back((int)p.seg.size());
        long long t = run.first;
        while (t < run.second) {
            const int r = (int)(t / tiles);
            const long long in_block = t - (long long)r * tiles;
            const long long stop = std::min<long long>(run.second - (long long)r * tiles, tiles);
            p.seg.push_back({r, (int)(in_block * etile), (int)std::min<long long>(N, stop * etile), 0});
            ++nseg_of_block[r];
            t = (long long)r * tiles + stop;
        }
    }
    p.cta_begin.push_back((int)p.seg.size());
    // slots: contiguous per receiver block, ordered by e_begin.  Runs are consecutive pieces of the flattened grid in
    // launch order, so the segments of one block appear in increasing e_begin.
    p.slot_begin.assign(p.rblocks + 1, 0);
    for (int r = 0; r < p.rblocks; ++r) p.slot_begin[r + 1] = p.slot_begin[r] + nseg_of_block[r];
    std::vector<int> next(p.slot_begin.begin(), p.slot_begin.end() - 1);
    for (Segment& sg : p.seg) sg.slot = next[sg.rblock]++;
    return p;
}

}  // namespace celes
