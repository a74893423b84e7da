// lbm_mesh.cuh — a1 in the paper's own form: voxelise a triangle mesh by axis-aligned ray casting (sm_100a).
//
// PAPER.md:191 "We re-voxelize the triangle mesh by casting axis-aligned rays through grid columns and computing
// ray-triangle intersections, using an odd-even parity rule along each column.  To improve robustness near degeneracies,
// we corroborate independent passes along different ray directions for solid labeling."  PAPER.md:51: ray-tracing-based
// occupancy test; Boolean merge with the base / terrain layers (done by voxelise_kernel, lbm_setup.cuh).
//
// Reading (DESIGN.md §4 reading 22), all in exact integer arithmetic so that the labels are unique and bit-exact against
// the oracle: vertices snapped to 1/256 cell (rint of float32 coord * 256), cell centres at (2i+1)*128.  Pass D casts
// rays along axis D; (u, v) = the other two axes in cyclic order.  A triangle is hit at P = (pu, pv) iff P is inside its
// (u,v) projection, taken counter-clockwise, with the top-left rule on the edges (P on edge a->b counts iff dv < 0, or
// dv == 0 and du > 0); zero-area projections are skipped.  The crossing w* flips every cell of the column whose centre
// is at or beyond it.  SOLID iff at least min_votes of the three passes end odd.
//
// Work decomposition: one WARP per triangle, lanes stride over the columns of its bounding box (a ground-sized triangle
// does not serialise in one thread); a hit toggles one byte (atomicXor on the enclosing word: XOR commutes, the result
// does not depend on the order); then one thread per column runs the prefix parity and adds it to the vote byte.
// Bit budget: coordinates in [-2^18, 2^19) -> differences < 2^20, edge functions and the doubled area < 2^41,
// |sum_i w_i z_i| < 2^62: int64 is exact.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace lbmk {

constexpr int MESH_SUB = 256;
constexpr int MESH_LO = -(1 << 18), MESH_HI = 1 << 19;

__device__ __forceinline__ long long floor_div(long long a, long long b) // b > 0
{
    long long q = a / b;
    return (a % b != 0 && a < 0) ? q - 1 : q;
}

template <int D>
__global__ void mesh_toggle_kernel(const float *__restrict__ tri, int ntri, uint32_t *__restrict__ toggles, int nx, int ny, int nz,
                                   int *__restrict__ err)
{
    constexpr int au = (D + 1) % 3, av = (D + 2) % 3, aw = D;
    const int warp = (int)((blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (warp >= ntri) return;
    const int n[3] = {nx, ny, nz};
    const int nu = n[au], nv = n[av], nw = n[aw];
    long long a[3], b[3], c[3];
    bool bad = false;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const float fa = tri[9 * (size_t)warp + k] * float(MESH_SUB), fb = tri[9 * (size_t)warp + 3 + k] * float(MESH_SUB),
                    fc = tri[9 * (size_t)warp + 6 + k] * float(MESH_SUB);
        bad |= !(fabsf(fa) < 1e9f && fabsf(fb) < 1e9f && fabsf(fc) < 1e9f); // also catches NaN
        a[k] = __float2int_rn(fa); b[k] = __float2int_rn(fb); c[k] = __float2int_rn(fc); // round half to even, as rint
        bad |= a[k] < MESH_LO || a[k] >= MESH_HI || b[k] < MESH_LO || b[k] >= MESH_HI || c[k] < MESH_LO || c[k] >= MESH_HI;
    }
    if (bad) { if (lane == 0) atomicExch(err, 1); return; }
    long long area = (b[au] - a[au]) * (c[av] - a[av]) - (b[av] - a[av]) * (c[au] - a[au]);
    if (area == 0) return;
    if (area < 0) {
#pragma unroll
        for (int k = 0; k < 3; ++k) { const long long t = b[k]; b[k] = c[k]; c[k] = t; }
        area = -area;
    }
    const long long umin = min(a[au], min(b[au], c[au])), umax = max(a[au], max(b[au], c[au]));
    const long long vmin = min(a[av], min(b[av], c[av])), vmax = max(a[av], max(b[av], c[av]));
    const long long iu0 = max(0LL, floor_div(umin - 128, 256)), iu1 = min((long long)nu - 1, floor_div(umax - 128, 256) + 1);
    const long long iv0 = max(0LL, floor_div(vmin - 128, 256)), iv1 = min((long long)nv - 1, floor_div(vmax - 128, 256) + 1);
    if (iu0 > iu1 || iv0 > iv1) return;
    const long long W = iu1 - iu0 + 1, total = W * (iv1 - iv0 + 1);
    // edge a->b: direction, inclusion of boundary points
    const long long d0u = c[au] - b[au], d0v = c[av] - b[av]; // edge b->c, weight of a
    const long long d1u = a[au] - c[au], d1v = a[av] - c[av]; // edge c->a, weight of b
    const long long d2u = b[au] - a[au], d2v = b[av] - a[av]; // edge a->b, weight of c
    const bool in0 = d0v < 0 || (d0v == 0 && d0u > 0), in1 = d1v < 0 || (d1v == 0 && d1u > 0), in2 = d2v < 0 || (d2v == 0 && d2u > 0);
    for (long long idx = lane; idx < total; idx += 32) {
        const long long iu = iu0 + idx % W, iv = iv0 + idx / W;
        const long long pu = (2 * iu + 1) * 128, pv = (2 * iv + 1) * 128;
        const long long wa = d0u * (pv - b[av]) - d0v * (pu - b[au]);
        const long long wb = d1u * (pv - c[av]) - d1v * (pu - c[au]);
        const long long wc = d2u * (pv - a[av]) - d2v * (pu - a[au]);
        if (!((wa > 0 || (wa == 0 && in0)) && (wb > 0 || (wb == 0 && in1)) && (wc > 0 || (wc == 0 && in2)))) continue;
        const long long num = wa * a[aw] + wb * b[aw] + wc * c[aw];
        const long long q = -floor_div(-num, 128 * area); // ceil(w* / 128)
        long long k = floor_div(q, 2);                    // first cell whose centre (2k+1) 128 >= w*
        if (k >= nw) continue;
        if (k < 0) k = 0;
        int xyz[3];
        xyz[au] = (int)iu; xyz[av] = (int)iv; xyz[aw] = (int)k;
        const long long cell = ((long long)xyz[2] * ny + xyz[1]) * nx + xyz[0];
        atomicXor(toggles + (cell >> 2), 1u << (8 * (int)(cell & 3)));
    }
}

// prefix parity along the rays of pass D, added to the votes
template <int D>
__global__ void mesh_scan_kernel(const uint8_t *__restrict__ toggles, uint8_t *__restrict__ votes, int nx, int ny, int nz)
{
    constexpr int au = (D + 1) % 3, av = (D + 2) % 3, aw = D;
    constexpr int ap = au < av ? au : av, aq = au < av ? av : au; // the lower-numbered axis runs fastest over the threads
    const int n[3] = {nx, ny, nz};
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= (long long)n[ap] * n[aq]) return;
    int xyz[3];
    xyz[ap] = (int)(t % n[ap]); xyz[aq] = (int)(t / n[ap]);
    unsigned par = 0;
    for (int k = 0; k < n[aw]; ++k) {
        xyz[aw] = k;
        const long long cell = ((long long)xyz[2] * ny + xyz[1]) * nx + xyz[0];
        par ^= toggles[cell] & 1u;
        votes[cell] = (uint8_t)(votes[cell] + par);
    }
}

} // namespace lbmk
