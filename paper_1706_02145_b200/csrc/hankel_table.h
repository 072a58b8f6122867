// hankel_table.h -- descriptor of the optional spherical-Hankel lookup table (host and device).
#pragma once
#include <cuda_runtime.h>

// Spherical-Hankel lookup table of the paper's scheme: node j holds, for p = 0..2 lmax,
// (Re h_p, Im h_p, dx Re h_p', dx Im h_p') at x_j = x0 + j dx; cubic Hermite interpolation between two nodes.
struct HankelTable {
    const float4* nodes;   // [n_nodes][P]
    float x0, inv_dx;
    int last;              // index of the last node
};
