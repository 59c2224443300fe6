// ORACLE — TEST INFRASTRUCTURE ONLY (see constants.hpp).
//
// Face-to-face grid traversal: the paper's `query` call returns "the index of the next cell, the pathlength to that
// cell" and propagation is "piece-wise linear integrations from cell face to cell face"
// (PAPER.md:209); BASELINE.json names it a 3D-DDA and asks for bit-exact cell-index sequences.  The paper prints no
// traversal algorithm, so this is the specification of DESIGN.md §"DDA", written once as a
// template: Real = float is the bit-exact reference for the GPU (compile with -ffp-contract=off: every multiply
// and add below is rounded on its own, no FMA), Real = double is the twin the oracle's walker uses.
//
// State: integer cell c[3], in-cell offset f[3] in the CLOSED interval [0,1] (cell units), direction k[3].
// One step:
//   per axis: k == 0 -> t = +inf;  else face = (k > 0 ? 1 : 0),  t = (face - f) * (1/k)   [one sub, one mul]
//   an axis that is periodic with extent 1 is treated as infinite: t = +inf and f is frozen (C3 note)
//   exit axis: x if t_x <= t_y and t_x <= t_z, else y if t_y <= t_z, else z          (ties: x before y before z)
//   segment length len = t_exit (>= 0, may be exactly 0)
//   other axes: f = clamp(f + len * k, 0, 1)   [one mul, one add]
//   exit axis:  f = (k > 0 ? 0 : 1);  c += sign(k);  wrap if periodic, else leaving the grid ends the ray.
#pragma once
#include <cstdint>
#include <limits>

namespace orc {

struct GridDims {
    int n[3];          // nx, ny, nz
    bool periodic[3];
    bool frozen(int ax) const { return periodic[ax] && n[ax] == 1; }
    int64_t linear(const int c[3]) const { return ((int64_t)c[2] * n[1] + c[1]) * (int64_t)n[0] + c[0]; }
};

template <class Real>
struct Ray {
    int c[3];
    Real f[3];
    Real k[3];
    Real inv[3];       // 1/k, set by set_direction
    void set_direction(const Real kk[3]) {
        for (int ax = 0; ax < 3; ++ax) { k[ax] = kk[ax]; inv[ax] = Real(1) / kk[ax]; }
    }
};

// Distance to the next face and the axis through which the ray leaves the current cell.
template <class Real>
inline int dda_next_face(const Ray<Real>& r, const GridDims& g, Real& len) {
    Real t[3];
    for (int ax = 0; ax < 3; ++ax) {
        if (r.k[ax] == Real(0) || g.frozen(ax)) {
            t[ax] = std::numeric_limits<Real>::infinity();
        } else {
            const Real face = r.k[ax] > Real(0) ? Real(1) : Real(0);
            const Real d = face - r.f[ax];
            t[ax] = d * r.inv[ax];
        }
    }
    int ex;
    if (t[0] <= t[1] && t[0] <= t[2]) ex = 0;
    else if (t[1] <= t[2]) ex = 1;
    else ex = 2;
    len = t[ex];
    return ex;
}

// Move a distance s (<= the distance to the next face) inside the current cell.
template <class Real>
inline void dda_advance_within(Ray<Real>& r, const GridDims& g, Real s) {
    for (int ax = 0; ax < 3; ++ax) {
        if (g.frozen(ax)) continue;
        const Real p = s * r.k[ax];
        Real nf = r.f[ax] + p;
        if (nf < Real(0)) nf = Real(0);
        if (nf > Real(1)) nf = Real(1);
        r.f[ax] = nf;
    }
}

// Cross the face found by dda_next_face.  Returns false if the ray left the grid through a non-periodic face.
template <class Real>
inline bool dda_cross(Ray<Real>& r, const GridDims& g, int ex, Real len) {
    for (int ax = 0; ax < 3; ++ax) {
        if (ax == ex || g.frozen(ax)) continue;
        const Real p = len * r.k[ax];
        Real nf = r.f[ax] + p;
        if (nf < Real(0)) nf = Real(0);
        if (nf > Real(1)) nf = Real(1);
        r.f[ax] = nf;
    }
    const int s = r.k[ex] > Real(0) ? 1 : -1;
    r.f[ex] = s > 0 ? Real(0) : Real(1);
    int cn = r.c[ex] + s;
    if (cn < 0 || cn >= g.n[ex]) {
        if (!g.periodic[ex]) return false;
        cn = cn < 0 ? g.n[ex] - 1 : 0;
    }
    r.c[ex] = cn;
    return true;
}

// Position in cell units -> (cell, offset): cell = floor(pos) clamped to [0, n-1], f = pos - cell (reading A20:
// a source exactly on a face belongs to the upper cell with f = 0).
template <class Real>
inline void dda_locate(Ray<Real>& r, const GridDims& g, const Real pos[3]) {
    for (int ax = 0; ax < 3; ++ax) {
        int c = (int)pos[ax];                       // pos >= 0: truncation == floor
        if (c > g.n[ax] - 1) c = g.n[ax] - 1;
        if (c < 0) c = 0;
        r.c[ax] = c;
        Real f = pos[ax] - (Real)c;
        if (f < Real(0)) f = Real(0);
        if (f > Real(1)) f = Real(1);
        r.f[ax] = f;
    }
}

}  // namespace orc
