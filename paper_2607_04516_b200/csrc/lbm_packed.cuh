// lbm_packed.cuh — the collision of lbm_core.cuh for TWO cells at once in packed FP32 pairs (sm_100a: add / sub / mul /
// fma.rn.f32x2 -> FADD2 / FMUL2 / FFMA2, one issue slot for two IEEE FP32 operations).  Same formulas, same operation
// order as collide() (DESIGN.md §3 steps 4b-4e); every packed operation rounds each half exactly as its scalar twin
// does, so the only differences to collide() are which multiply-adds are fused (here: the ones written as fma2).  The
// division and the square roots have no packed form and run per cell.  Used by the two-cells-per-thread launch shape
// (lbm_step_vec.cuh, V = 2), whose 2 x 241 scalar FP32 instructions per thread become ~300.
#pragma once
#include "lbm_core.cuh"

namespace lbmk {

struct f2 { unsigned long long v; }; // {lo = cell 0, hi = cell 1}

__device__ __forceinline__ f2 pk(float a, float b) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ f2 bc(float a) { return pk(a, a); }
__device__ __forceinline__ void upk(f2 a, float &x, float &y) { asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(a.v)); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ f2 sub2(f2 a, f2 b) { f2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return r; }

// c . a for a pair vector known at compile time (pair vectors have c_x >= 0 and a positive first non-zero component)
template <int CX, int CY, int CZ>
__device__ __forceinline__ f2 cdot2(f2 ax, f2 ay, f2 az)
{
    static_assert(CX >= 0 && (CX != 0 || CY >= 0) && (CX != 0 || CY != 0 || CZ > 0), "pair vectors only");
    if constexpr (CX != 0 && CY == 0 && CZ == 0) return ax;
    else if constexpr (CX == 0 && CY != 0 && CZ == 0) return ay;
    else if constexpr (CX == 0 && CY == 0) return az;
    else if constexpr (CZ == 0) return CY > 0 ? add2(ax, ay) : sub2(ax, ay);
    else if constexpr (CY == 0) return CZ > 0 ? add2(ax, az) : sub2(ax, az);
    else return CZ > 0 ? add2(ay, az) : sub2(ay, az);
}

// In: pulled populations of two cells.  Out: their post-collision populations and the (rho, u) each collision used.
__device__ __forceinline__ void collide2(float (&ga)[Q], float (&gb)[Q], const Params<float> &P, Macro<float> &ma, Macro<float> &mb)
{
    f2 g[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) g[i] = pk(ga[i], gb[i]);
    f2 s[10], d[10];
#pragma unroll
    for (int k = 1; k <= 9; ++k) { s[k] = add2(g[2 * k - 1], g[2 * k]); d[k] = sub2(g[2 * k - 1], g[2 * k]); }
    // 4b
    const f2 drho = add2(g[0], add2(add2(add2(add2(s[1], s[2]), add2(s[3], s[4])), add2(add2(s[5], s[6]), add2(s[7], s[8]))), s[9]));
    const f2 mx = add2(add2(add2(d[1], d[4]), add2(d[5], d[7])), d[8]);
    const f2 my = add2(add2(add2(d[2], d[4]), sub2(d[6], d[7])), d[9]);
    const f2 mz = sub2(add2(add2(d[3], d[5]), sub2(d[6], d[8])), d[9]);
    const f2 Mxx = add2(add2(add2(s[1], s[4]), add2(s[5], s[7])), s[8]);
    const f2 Myy = add2(add2(add2(s[2], s[4]), add2(s[6], s[7])), s[9]);
    const f2 Mzz = add2(add2(add2(s[3], s[5]), add2(s[6], s[8])), s[9]);
    const f2 Mxy = sub2(s[4], s[7]), Mxz = sub2(s[5], s[8]), Myz = sub2(s[6], s[9]);
    const f2 rho = add2(drho, bc(1.0f));
    float r0, r1;
    upk(rho, r0, r1);
    const f2 inv = pk(1.0f / r0, 1.0f / r1);
    // 4c: u = (b - h x b + h (h.b)) / (1 + |h|^2), b = m/rho + F/2
    const f2 bx = fma2(mx, inv, bc(0.5f * P.Fx)), by = fma2(my, inv, bc(0.5f * P.Fy)), bz = fma2(mz, inv, bc(0.5f * P.Fz));
    const f2 hb = fma2(bc(P.hx), bx, fma2(bc(P.hy), by, mul2(bc(P.hz), bz)));
    const f2 i1 = bc(P.inv1ph2);
    const f2 ux = mul2(fma2(bc(P.hx), hb, fma2(bc(P.hz), by, fma2(bc(-P.hy), bz, bx))), i1);
    const f2 uy = mul2(fma2(bc(P.hy), hb, fma2(bc(P.hx), bz, fma2(bc(-P.hz), bx, by))), i1);
    const f2 uz = mul2(fma2(bc(P.hz), hb, fma2(bc(P.hy), bx, fma2(bc(-P.hx), by, bz))), i1);
    // Fd = rho (F - f x u)
    const f2 Fdx = mul2(rho, fma2(bc(P.fz), uy, fma2(bc(-P.fy), uz, bc(P.Fx))));
    const f2 Fdy = mul2(rho, fma2(bc(P.fx), uz, fma2(bc(-P.fz), ux, bc(P.Fy))));
    const f2 Fdz = mul2(rho, fma2(bc(P.fy), ux, fma2(bc(-P.fx), uy, bc(P.Fz))));
    // 4d: Pi = M - (drho/3) I - rho u u
    const f2 nrho = sub2(bc(0.0f), rho);
    const f2 nrux = mul2(nrho, ux), nruy = mul2(nrho, uy), nruz = mul2(nrho, uz);
    const f2 t3 = mul2(drho, bc(-1.0f / 3.0f));
    const f2 Pxx = fma2(nrux, ux, add2(Mxx, t3)), Pyy = fma2(nruy, uy, add2(Myy, t3)), Pzz = fma2(nruz, uz, add2(Mzz, t3));
    const f2 Pxy = fma2(nrux, uy, Mxy), Pxz = fma2(nrux, uz, Mxz), Pyz = fma2(nruy, uz, Myz);
    const f2 q2 = fma2(fma2(Pxy, Pxy, fma2(Pxz, Pxz, mul2(Pyz, Pyz))), bc(2.0f), fma2(Pxx, Pxx, fma2(Pyy, Pyy, mul2(Pzz, Pzz))));
    float q0, q1;
    upk(q2, q0, q1);
    const f2 Qn = pk(sqrtf(q0), sqrtf(q1));
    const f2 arg = fma2(mul2(bc(P.Kles), Qn), inv, bc(P.tau0 * P.tau0));
    float a0, a1;
    upk(arg, a0, a1);
    const f2 tau = fma2(pk(sqrtf(a0), sqrtf(a1)), bc(0.5f), bc(0.5f * P.tau0));
    float t0, t1;
    upk(tau, t0, t1);
    const f2 omega = pk(1.0f / t0, 1.0f / t1);
    const f2 phi = fma2(omega, bc(-0.5f), bc(1.0f));
    // 4e (see collide() for the expansion)
    const f2 uF = fma2(ux, Fdx, fma2(uy, Fdy, mul2(uz, Fdz)));
    const f2 uu = fma2(ux, ux, fma2(uy, uy, mul2(uz, uz)));
    const f2 A0 = fma2(mul2(nrho, bc(1.5f)), uu, drho);
    const f2 keep = sub2(bc(1.0f), omega);
    const f2 base = fma2(omega, A0, mul2(mul2(phi, bc(-3.0f)), uF));
    const f2 orho = mul2(omega, rho);
    const f2 P1x = mul2(orho, ux), P1y = mul2(orho, uy), P1z = mul2(orho, uz);
    const f2 P2x = mul2(phi, Fdx), P2y = mul2(phi, Fdy), P2z = mul2(phi, Fdz);
    g[0] = fma2(keep, g[0], mul2(base, bc(1.0f / 3.0f)));
    const f2 E0a = mul2(base, bc(1.0f / 18.0f)), E0b = mul2(base, bc(1.0f / 36.0f));
    const f2 vax = fma2(P1x, bc(0.25f), mul2(P2x, bc(0.5f))), vay = fma2(P1y, bc(0.25f), mul2(P2y, bc(0.5f))), vaz = fma2(P1z, bc(0.25f), mul2(P2z, bc(0.5f)));
    const f2 oax = mul2(add2(P1x, P2x), bc(1.0f / 6.0f)), oay = mul2(add2(P1y, P2y), bc(1.0f / 6.0f)), oaz = mul2(add2(P1z, P2z), bc(1.0f / 6.0f));
    const f2 vbx = mul2(vax, bc(0.5f)), vby = mul2(vay, bc(0.5f)), vbz = mul2(vaz, bc(0.5f));
    const f2 obx = mul2(oax, bc(0.5f)), oby = mul2(oay, bc(0.5f)), obz = mul2(oaz, bc(0.5f));
    static_for<1, 10>([&](auto kc) {
        constexpr int k = decltype(kc)::value;
        constexpr int cx = pair_cx(k), cy = pair_cy(k), cz = pair_cz(k);
        const f2 E0 = (k <= 3) ? E0a : E0b;
        const f2 cu = cdot2<cx, cy, cz>(ux, uy, uz);
        const f2 cv = (k <= 3) ? cdot2<cx, cy, cz>(vax, vay, vaz) : cdot2<cx, cy, cz>(vbx, vby, vbz);
        const f2 co = (k <= 3) ? cdot2<cx, cy, cz>(oax, oay, oaz) : cdot2<cx, cy, cz>(obx, oby, obz);
        const f2 even = fma2(cu, cv, E0);
        g[2 * k - 1] = fma2(keep, g[2 * k - 1], add2(even, co));
        g[2 * k] = fma2(keep, g[2 * k], sub2(even, co));
    });
#pragma unroll
    for (int i = 0; i < Q; ++i) upk(g[i], ga[i], gb[i]);
    float ua, ub;
    ma.rho = r0; mb.rho = r1;
    upk(ux, ua, ub); ma.ux = ua; mb.ux = ub;
    upk(uy, ua, ub); ma.uy = ua; mb.uy = ub;
    upk(uz, ua, ub); ma.uz = ua; mb.uz = ub;
}

} // namespace lbmk
