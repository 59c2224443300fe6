// a4 DDA cell march — the paper's `query`: "index of the next cell, the pathlength to that cell",
// propagation "from cell face to cell face".  The paper prints no traversal algorithm; this is the
// specification of DESIGN.md §DDA, in fp32 with every multiply/add/subtract/divide rounded on its own
// (__fmul_rn / __fadd_rn / __fsub_rn / __fdiv_rn are never contracted into FMAs), so that the sequence of cells is
// bit-exact against any IEEE-754 implementation of the same specification.
//
// State: integer cell c, in-cell offset f in the CLOSED interval [0,1] (cell units), direction k, inv = 1/k.
//   per axis: k == 0 or frozen axis -> t = +inf; else face = (k > 0 ? 1 : 0), t = (face - f) * inv
//   exit axis: x if t_x <= t_y and t_x <= t_z, else y if t_y <= t_z, else z; segment length = t_exit
//   other axes: f = clamp(f + len * k, 0, 1);  exit axis: f = (k > 0 ? 0 : 1), c += sign(k), wrap or leave.
// A periodic axis of extent 1 is "frozen": treated as infinite, its offset never changes.
#pragma once
#include <cstdint>
#include <math_constants.h>

namespace thor {

struct GridDims {
    int nx, ny, nz;
    unsigned periodic;   // bit 0,1,2 = x,y,z
    unsigned frozen;     // bit 0,1,2: periodic with extent 1
};

struct Ray {
    int cx, cy, cz;
    float fx, fy, fz;
    float kx, ky, kz;
    float ix, iy, iz;    // 1/k, correctly rounded (__frcp_rn: the same value as the IEEE quotient 1/k, in fewer instructions)
};

__device__ __forceinline__ void ray_set_direction(Ray& r, float kx, float ky, float kz) {
    r.kx = kx; r.ky = ky; r.kz = kz;
    r.ix = __frcp_rn(kx); r.iy = __frcp_rn(ky); r.iz = __frcp_rn(kz);
}

// Direction now, reciprocals later: a packet that scatters deep inside a cell never needs them (walk_kernel).
__device__ __forceinline__ void ray_set_k(Ray& r, float kx, float ky, float kz) { r.kx = kx; r.ky = ky; r.kz = kz; }
__device__ __forceinline__ void ray_set_inv(Ray& r) {
    r.ix = __frcp_rn(r.kx); r.iy = __frcp_rn(r.ky); r.iz = __frcp_rn(r.kz);
}

// Distance from the in-cell position to the nearest face of the cell in ANY direction (frozen axes have none): a
// lower bound of the segment length dda_next_face would return, at the cost of six min operations.
__device__ __forceinline__ float dda_min_face_distance(const Ray& r, const GridDims& g) {
    const float dx = (g.frozen & 1u) ? CUDART_INF_F : fminf(r.fx, 1.0f - r.fx);
    const float dy = (g.frozen & 2u) ? CUDART_INF_F : fminf(r.fy, 1.0f - r.fy);
    const float dz = (g.frozen & 4u) ? CUDART_INF_F : fminf(r.fz, 1.0f - r.fz);
    return fminf(dx, fminf(dy, dz));
}

__device__ __forceinline__ float dda_t_axis(float f, float k, float inv, bool frozen) {
    const float face = k > 0.0f ? 1.0f : 0.0f;
    const float t = __fmul_rn(__fsub_rn(face, f), inv);
    return (k == 0.0f || frozen) ? CUDART_INF_F : t;
}

// Distance to the next face; returns the exit axis (0,1,2).
__device__ __forceinline__ int dda_next_face(const Ray& r, const GridDims& g, float& len) {
    const float tx = dda_t_axis(r.fx, r.kx, r.ix, g.frozen & 1u);
    const float ty = dda_t_axis(r.fy, r.ky, r.iy, g.frozen & 2u);
    const float tz = dda_t_axis(r.fz, r.kz, r.iz, g.frozen & 4u);
    int ex;
    if (tx <= ty && tx <= tz) { ex = 0; len = tx; }
    else if (ty <= tz) { ex = 1; len = ty; }
    else { ex = 2; len = tz; }
    return ex;
}

__device__ __forceinline__ float dda_move(float f, float s, float k) {
    const float nf = __fadd_rn(f, __fmul_rn(s, k));
    return fminf(fmaxf(nf, 0.0f), 1.0f);
}

// Move a distance s (<= distance to the next face) inside the current cell.
__device__ __forceinline__ void dda_advance_within(Ray& r, const GridDims& g, float s) {
    if (!(g.frozen & 1u)) r.fx = dda_move(r.fx, s, r.kx);
    if (!(g.frozen & 2u)) r.fy = dda_move(r.fy, s, r.ky);
    if (!(g.frozen & 4u)) r.fz = dda_move(r.fz, s, r.kz);
}

// Cross the face found by dda_next_face.  Returns false if the ray left the grid through a non-periodic face.
// Written with selects only: the exit axis differs from lane to lane, and per-axis branches would run each axis with a third
// of the warp (measured on the thin `gather` workload: 20 % of the kernel's issued instructions at 6-13 of 32 lanes).
__device__ __forceinline__ bool dda_cross(Ray& r, const GridDims& g, int ex, float len) {
    const float mx = (g.frozen & 1u) ? r.fx : dda_move(r.fx, len, r.kx);      // warp-uniform conditions
    const float my = (g.frozen & 2u) ? r.fy : dda_move(r.fy, len, r.ky);
    const float mz = (g.frozen & 4u) ? r.fz : dda_move(r.fz, len, r.kz);
    const float ke = ex == 0 ? r.kx : ex == 1 ? r.ky : r.kz;
    const int n = ex == 0 ? g.nx : ex == 1 ? g.ny : g.nz;
    const int s = ke > 0.0f ? 1 : -1;
    const float fe = s > 0 ? 0.0f : 1.0f;
    int c = (ex == 0 ? r.cx : ex == 1 ? r.cy : r.cz) + s;
    const bool out = c < 0 || c >= n;
    const bool wrap = (g.periodic & (1u << ex)) != 0u;
    c = (out && wrap) ? (c < 0 ? n - 1 : 0) : c;
    const bool inside = !out || wrap;
    // the exit axis lands on the face of the new cell (only if there is one); the other axes move by len unless frozen
    r.fx = ex == 0 ? (inside ? fe : r.fx) : mx;
    r.fy = ex == 1 ? (inside ? fe : r.fy) : my;
    r.fz = ex == 2 ? (inside ? fe : r.fz) : mz;
    r.cx = (inside && ex == 0) ? c : r.cx;
    r.cy = (inside && ex == 1) ? c : r.cy;
    r.cz = (inside && ex == 2) ? c : r.cz;
    return inside;
}

// Position in cell units -> (cell, offset): cell = floor(pos) clamped to [0, n-1], f = pos - cell clamped to [0,1]
// (reading A20: a source exactly on a face belongs to the upper cell with f = 0).
__device__ __forceinline__ void dda_locate_axis(float pos, int n, int& c, float& f) {
    int ci = (int)pos;
    ci = min(max(ci, 0), n - 1);
    c = ci;
    f = fminf(fmaxf(__fsub_rn(pos, (float)ci), 0.0f), 1.0f);
}

__device__ __forceinline__ void dda_locate(Ray& r, const GridDims& g, float px, float py, float pz) {
    dda_locate_axis(px, g.nx, r.cx, r.fx);
    dda_locate_axis(py, g.ny, r.cy, r.fy);
    dda_locate_axis(pz, g.nz, r.cz, r.fz);
}

__device__ __forceinline__ int64_t dda_linear(const Ray& r, const GridDims& g) {
    return ((int64_t)r.cz * g.ny + r.cy) * (int64_t)g.nx + r.cx;
}

// The same specification for a ray whose direction never changes (ray-tracing operators): everything that depends on k
// alone is folded into per-axis constants once, so a step is 6 flops for the face distances, one compare chain, and per
// axis one multiply, one saturating add and one select.  Same cells, same segment lengths as dda_next_face / dda_cross:
//   dead axis (k == 0 or frozen): face = +inf, inv = 1 -> t = (inf - f) * 1 = +inf;  frozen: k_move = 0 -> f unchanged
//   clamp(x, 0, 1) is __saturatef(x) (NaN -> 0 as fminf(fmaxf(NaN, 0), 1) does)
// The march ends at the first box face, periodic or not (thor_raytrace's contract), so there is no wrap.
struct RayMarch {
    float fx, fy, fz;          // in-cell offsets
    float ax, ay, az;          // face coordinate 1 / 0, or +inf on a dead axis
    float ix, iy, iz;          // 1/k, or 1 on a dead axis
    float kx, ky, kz;          // k, or 0 on a frozen axis (offset never changes)
    float ex, ey, ez;          // offset on entering the next cell along the axis: 0 (k > 0) or 1
    int cx, cy, cz;            // cell
    int sx, sy, sz;            // sign(k) as the cell step
    int64_t dy, dz;            // signed strides of y and z in the linear index (x: sx)
    int64_t idx;               // linear index of the cell
};

__device__ __forceinline__ void march_init(RayMarch& m, const GridDims& g, float px, float py, float pz, float kx,
                                           float ky, float kz) {
    dda_locate_axis(px, g.nx, m.cx, m.fx);
    dda_locate_axis(py, g.ny, m.cy, m.fy);
    dda_locate_axis(pz, g.nz, m.cz, m.fz);
    const bool dx = kx == 0.0f || (g.frozen & 1u), dy = ky == 0.0f || (g.frozen & 2u), dz = kz == 0.0f || (g.frozen & 4u);
    m.ax = dx ? CUDART_INF_F : (kx > 0.0f ? 1.0f : 0.0f);
    m.ay = dy ? CUDART_INF_F : (ky > 0.0f ? 1.0f : 0.0f);
    m.az = dz ? CUDART_INF_F : (kz > 0.0f ? 1.0f : 0.0f);
    m.ix = dx ? 1.0f : __frcp_rn(kx);
    m.iy = dy ? 1.0f : __frcp_rn(ky);
    m.iz = dz ? 1.0f : __frcp_rn(kz);
    m.kx = (g.frozen & 1u) ? 0.0f : kx;
    m.ky = (g.frozen & 2u) ? 0.0f : ky;
    m.kz = (g.frozen & 4u) ? 0.0f : kz;
    m.ex = kx > 0.0f ? 0.0f : 1.0f; m.ey = ky > 0.0f ? 0.0f : 1.0f; m.ez = kz > 0.0f ? 0.0f : 1.0f;
    m.sx = kx > 0.0f ? 1 : -1; m.sy = ky > 0.0f ? 1 : -1; m.sz = kz > 0.0f ? 1 : -1;
    m.dy = (int64_t)m.sy * g.nx;
    m.dz = (int64_t)m.sz * g.nx * g.ny;
    m.idx = ((int64_t)m.cz * g.ny + m.cy) * (int64_t)g.nx + m.cx;
}

// Segment length through the current cell and the exit axis as two predicates (x, y; else z).
__device__ __forceinline__ float march_next_face(const RayMarch& m, bool& ex_x, bool& ex_y) {
    const float tx = __fmul_rn(__fsub_rn(m.ax, m.fx), m.ix);
    const float ty = __fmul_rn(__fsub_rn(m.ay, m.fy), m.iy);
    const float tz = __fmul_rn(__fsub_rn(m.az, m.fz), m.iz);
    ex_x = tx <= ty && tx <= tz;
    ex_y = !ex_x && ty <= tz;
    return ex_x ? tx : ex_y ? ty : tz;
}

// Cross the exit face; false if the ray left the box.
__device__ __forceinline__ bool march_cross(RayMarch& m, const GridDims& g, bool ex_x, bool ex_y, float len) {
    const bool ex_z = !ex_x && !ex_y;
    const float nx = __saturatef(__fadd_rn(m.fx, __fmul_rn(len, m.kx)));
    const float ny = __saturatef(__fadd_rn(m.fy, __fmul_rn(len, m.ky)));
    const float nz = __saturatef(__fadd_rn(m.fz, __fmul_rn(len, m.kz)));
    m.fx = ex_x ? m.ex : nx;                                   // the exit axis is never dead: entry offset 0 / 1 by sign(k)
    m.fy = ex_y ? m.ey : ny;
    m.fz = ex_z ? m.ez : nz;
    if (ex_x) { m.cx += m.sx; m.idx += m.sx; }
    if (ex_y) { m.cy += m.sy; m.idx += m.dy; }
    if (ex_z) { m.cz += m.sz; m.idx += m.dz; }
    return (unsigned)m.cx < (unsigned)g.nx && (unsigned)m.cy < (unsigned)g.ny && (unsigned)m.cz < (unsigned)g.nz;
}

// The same crossing for a sight line that wraps at periodic faces: an exit through a periodic face re-enters
// at the opposite one (cell and linear index wrapped); a non-periodic face ends the ray as above.
__device__ __forceinline__ bool march_cross_wrap(RayMarch& m, const GridDims& g, bool ex_x, bool ex_y, float len) {
    if (march_cross(m, g, ex_x, ex_y, len)) return true;
    const bool ex_z = !ex_x && !ex_y;
    if (ex_x && (g.periodic & 1u)) { const int w = m.cx < 0 ? g.nx : -g.nx; m.cx += w; m.idx += w; return true; }
    if (ex_y && (g.periodic & 2u)) { const int w = m.cy < 0 ? g.ny : -g.ny; m.cy += w; m.idx += (int64_t)w * g.nx; return true; }
    if (ex_z && (g.periodic & 4u)) { const int w = m.cz < 0 ? g.nz : -g.nz; m.cz += w; m.idx += (int64_t)w * g.nx * g.ny; return true; }
    return false;
}

}  // namespace thor
