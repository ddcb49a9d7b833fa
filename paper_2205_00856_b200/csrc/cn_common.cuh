// Common device helpers: complex128 arithmetic written out in re/im with explicit FMAs
// (the paper notes the same hand expansion paid off on its GPU), and the
// first-order linear recurrence scan used by every sweep.
//
// Scaled system: every row of Eq. 5 is multiplied by kappa = i / s with
// s = dt / (4 dx^2).  Because b = c = -i s this makes both off-diagonals of kappa*T exactly 1 and
// its diagonal mu_j = -gamma_j + i rho,  gamma_j = 2 + 2 dx^2 V_j,  rho = 1 / s = 4 dx^2 / dt.
// The scaled right-hand side of Eq. 3 is E_j = (gamma_j + i rho) psi_j - psi_{j-1} - psi_{j+1}.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

typedef double2 cplx;

#define CN_DEVINL __device__ __forceinline__

CN_DEVINL cplx cmake(double x, double y) { return make_double2(x, y); }
CN_DEVINL cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
CN_DEVINL cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
CN_DEVINL cplx cneg(cplx a) { return make_double2(-a.x, -a.y); }
CN_DEVINL cplx cmul(cplx a, cplx b)
{
    return make_double2(fma(-a.y, b.y, a.x * b.x), fma(a.y, b.x, a.x * b.y));
}
// c + a*b
CN_DEVINL cplx cfma(cplx a, cplx b, cplx c)
{
    return make_double2(fma(-a.y, b.y, fma(a.x, b.x, c.x)), fma(a.y, b.x, fma(a.x, b.y, c.y)));
}
// c - a*b
CN_DEVINL cplx cfnma(cplx a, cplx b, cplx c)
{
    return make_double2(fma(a.y, b.y, fma(-a.x, b.x, c.x)), fma(-a.y, b.x, fma(-a.x, b.y, c.y)));
}
// a*b - c
CN_DEVINL cplx cmsub(cplx a, cplx b, cplx c)
{
    return make_double2(fma(-a.y, b.y, fma(a.x, b.x, -c.x)), fma(a.y, b.x, fma(a.x, b.y, -c.y)));
}
CN_DEVINL cplx crecip(cplx a)
{
    // scaled by the larger component so that |a|^2 can neither overflow nor underflow early
    double m = fmax(fabs(a.x), fabs(a.y));
    double inv_m = 1.0 / m;
    double xr = a.x * inv_m, xi = a.y * inv_m;
    double d = 1.0 / (fma(xr, xr, xi * xi));
    return make_double2(xr * d * inv_m, -xi * d * inv_m);
}
// the same with ONE division when |a|^2 can neither overflow nor underflow (the factor kernels: ~10 reciprocals per thread)
CN_DEVINL cplx crecip_fast(cplx a)
{
    const double m = fmax(fabs(a.x), fabs(a.y));
    if (m > 1e-140 && m < 1e140) {
        const double d = 1.0 / fma(a.x, a.x, a.y * a.y);
        return make_double2(a.x * d, -a.y * d);
    }
    return crecip(a);
}
// 1 / m for a positive, normal m: hardware seed (rcp.approx.ftz.f64, ~20 bits over the whole exponent range) and two
// Newton steps -- five instructions, no branch, within an ulp or two of the correctly rounded quotient (a division
// compiles to ~25 instructions with a slow-path call)
CN_DEVINL double rcp_pos(double m)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(m));
    double e = fma(-m, r, 1.0);
    r = fma(r, e, r);
    e = fma(-m, r, 1.0);
    return fma(r, e, r);
}
CN_DEVINL bool cfinite_nonzero(cplx a)
{
    return isfinite(a.x) && isfinite(a.y) && (a.x != 0.0 || a.y != 0.0);
}

// E = (gamma + i rho) * p - lo - hi      (scaled Eq. 3)
CN_DEVINL cplx rhs_E(double gamma, double rho, cplx p, cplx lo, cplx hi)
{
    double er = fma(gamma, p.x, fma(-rho, p.y, -(lo.x + hi.x)));
    double ei = fma(gamma, p.y, fma(rho, p.x, -(lo.y + hi.y)));
    return make_double2(er, ei);
}

// Programmatic dependent launch (sm_90+): every kernel of the per-step chain is launched with
// programmatic stream serialization, fetches what does not depend on its predecessor, then waits for the
// predecessor to COMPLETE (memory flushed) with pdl_wait().  Because every kernel of the chain executes
// pdl_wait() before it finishes, completion is transitive: after pdl_wait() all earlier kernels are done.
// Without the launch attribute both instructions are no-ops.
CN_DEVINL void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
CN_DEVINL void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Load of a value the PRECEDING kernel of the chain produced, used after pdl_wait().  The pointers of the RS kernels
// are `const __restrict__`, which allows the compiler to turn a plain load into ld.global.nc and to hoist it above
// the wait; a volatile asm with a memory clobber stays below it and reads through L2.
CN_DEVINL cplx ld_dep(const cplx *p)
{
    cplx v;
    asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}

CN_DEVINL cplx shfl_up_c(cplx v, int d)
{
    return make_double2(__shfl_up_sync(0xffffffffu, v.x, d), __shfl_up_sync(0xffffffffu, v.y, d));
}
CN_DEVINL cplx shfl_down_c(cplx v, int d)
{
    return make_double2(__shfl_down_sync(0xffffffffu, v.x, d), __shfl_down_sync(0xffffffffu, v.y, d));
}
CN_DEVINL cplx shfl_c(cplx v, int src)
{
    return make_double2(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}

// ---- scan of affine maps  x -> A x + B  ------------------------------------------------------------
// A sweep D_i = E_i - q_{i-1} D_{i-1} restricted to one thread's chunk is the affine map
// "value entering the chunk -> value leaving it".  Composing the maps of consecutive chunks gives
// every chunk its true inflow.  At a joint line the value is reset, i.e. A = 0, which is what keeps
// blocks independent ("no communication at this stage").
//
// Warp-level inclusive Kogge-Stone over lanes in direction DIR (+1: information flows to higher
// lanes, -1: to lower lanes).  STEPS = number of doubling steps (5 for a full warp; fewer when a
// block spans fewer than 32 chunks, because A = 0 at block ends makes later steps no-ops).
template <int DIR, int STEPS>
CN_DEVINL void warp_scan_affine(cplx &A, cplx &B, int lane)
{
#pragma unroll
    for (int k = 0; k < STEPS; ++k) {
        const int d = 1 << k;
        cplx As = (DIR > 0) ? shfl_up_c(A, d) : shfl_down_c(A, d);
        cplx Bs = (DIR > 0) ? shfl_up_c(B, d) : shfl_down_c(B, d);
        bool ok = (DIR > 0) ? (lane >= d) : (lane + d < 32);
        if (ok) {
            B = cfma(A, Bs, B);
            A = cmul(A, As);
        }
    }
}

// The same scan without the lane predicate.  Valid when A = 0 at the FIRST element of every chain in direction DIR
// (a lane whose prefix already starts at its chain's first element then has A = 0, so combining it with whatever the
// out-of-range or foreign lane holds leaves B unchanged): saves the compare and the selects of every step.
template <int DIR, int STEPS>
CN_DEVINL void warp_scan_affine_uncond(cplx &A, cplx &B)
{
#pragma unroll
    for (int k = 0; k < STEPS; ++k) {
        const int d = 1 << k;
        cplx As = (DIR > 0) ? shfl_up_c(A, d) : shfl_down_c(A, d);
        cplx Bs = (DIR > 0) ? shfl_up_c(B, d) : shfl_down_c(B, d);
        B = cfma(A, Bs, B);
        A = cmul(A, As);
    }
}
