// partition.h -- host side of the block-diagonal preconditioner: division of the sphere set into subsets G_j
// by an array of cuboids (step 1 of section 3.2.1; Fig. 1).
//
// The cuboid array is anchored at the minimum corner of the bounding box of the centres; sphere i falls into
// cell (floor((x_i - x_min)/e_x), floor((y_i - y_min)/e_y), floor((z_i - z_min)/e_z)).  Non-empty cells are
// numbered in lexicographic (cx, cy, cz) order; inside a cell spheres keep their index order.  The paper
// renumbers the spheres so that a subset is a run of successive indices; here the vectors keep the caller's
// order and `order` is that renumbering (subset j = order[offset[j]] .. order[offset[j+1]-1]).
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

namespace celes {

struct Partition {
    std::vector<int> order;      // [N] sphere indices sorted by subset
    std::vector<int> offset;     // [n_groups + 1]
    std::vector<int> group_of;   // [N] subset of sphere i
    int n_groups() const { return (int)offset.size() - 1; }
    int max_group() const {
        int m = 0;
        for (size_t j = 0; j + 1 < offset.size(); ++j) m = std::max(m, offset[j + 1] - offset[j]);
        return m;
    }
};

// edge[a] <= 0 or non-finite means "do not cut along axis a".  Returns false on invalid input.
inline bool build_partition(int N, const double* pos, const double edge[3], Partition& out) {
    if (N < 1 || !pos) return false;
    double lo[3] = {pos[0], pos[1], pos[2]};
    for (int i = 0; i < N; ++i)
        for (int a = 0; a < 3; ++a) {
            if (!std::isfinite(pos[3 * i + a])) return false;
            lo[a] = std::min(lo[a], pos[3 * i + a]);
        }
    struct Key { int64_t c[3]; int i; };
    std::vector<Key> keys(N);
    for (int i = 0; i < N; ++i) {
        for (int a = 0; a < 3; ++a) {
            const bool cut = std::isfinite(edge[a]) && edge[a] > 0.0;
            keys[i].c[a] = cut ? (int64_t)std::floor((pos[3 * i + a] - lo[a]) / edge[a]) : 0;
        }
        keys[i].i = i;
    }
    std::sort(keys.begin(), keys.end(), [](const Key& x, const Key& y) {
        if (x.c[0] != y.c[0]) return x.c[0] < y.c[0];
        if (x.c[1] != y.c[1]) return x.c[1] < y.c[1];
        if (x.c[2] != y.c[2]) return x.c[2] < y.c[2];
        return x.i < y.i;
    });
    out.order.resize(N);
    out.group_of.resize(N);
    out.offset.clear();
    for (int t = 0; t < N; ++t) {
        const bool first = t == 0 || keys[t].c[0] != keys[t - 1].c[0] || keys[t].c[1] != keys[t - 1].c[1] ||
                           keys[t].c[2] != keys[t - 1].c[2];
        if (first) out.offset.push_back(t);
        out.order[t] = keys[t].i;
        out.group_of[keys[t].i] = (int)out.offset.size() - 1;
    }
    out.offset.push_back(N);
    return true;
}

}  // namespace celes
