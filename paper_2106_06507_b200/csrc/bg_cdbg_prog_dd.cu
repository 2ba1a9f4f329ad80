// Double-double instantiation of the colour-class program interpreter (bg_cdbg_interp.cuh): the re-evaluation of
// the events the FP64 interpreter flagged as ill-conditioned (BG_OPT_PRECISION = 2).
// Same class programs, same event records, same state offsets - a state element is a complex double-double
// (32 bytes) instead of a complex double, so half as much of the state fits in shared memory.
#include "bg_ddmath.cuh"
#include "bg_cdbg_interp.cuh"

namespace bg {

struct alignas(16) dd4 { double2 a, b; };   // (re.hi, re.lo), (im.hi, im.lo)

template <> struct StateElem<cxd> {
    using T = dd4;
    using R = dd;
    static constexpr bool kComplex = true, kDD = true;
    static __device__ __forceinline__ cxd get(dd4 v) { return mkd(mkdd(v.a.x, v.a.y), mkdd(v.b.x, v.b.y)); }
    static __device__ __forceinline__ dd4 put(cxd v) {
        dd4 r;
        r.a = make_double2(v.re.hi, v.re.lo);
        r.b = make_double2(v.im.hi, v.im.lo);
        return r;
    }
    static __device__ __forceinline__ cxd make(dd re, dd im) { return mkd(re, im); }
    static __device__ __forceinline__ dd4 ldcg(const dd4* p) {
        dd4 r;
        r.a = __ldcg(&p->a);
        r.b = __ldcg(&p->b);
        return r;
    }
    static __device__ __forceinline__ void stcg(dd4* p, dd4 v) {
        __stcg(&p->a, v.a);
        __stcg(&p->b, v.b);
    }
};

__device__ __forceinline__ dd r_add(dd a, dd b) { return dd_add(a, b); }
__device__ __forceinline__ dd r_sub(dd a, dd b) { return dd_sub(a, b); }
__device__ __forceinline__ dd r_from(double x, dd) { return mkdd(x); }
__device__ __forceinline__ double r_hi(dd x) { return x.hi; }
// 1/sqrt2 to 106 bits
__device__ __forceinline__ dd dd_isqrt2() { return mkdd(0.70710678118654757, -4.8336466567264567e-17); }
__device__ __forceinline__ cxd s_isqrt2(cxd v) { return cxd_scale(dd_isqrt2(), v); }
__device__ __forceinline__ dd r_isqrt2_over(dd p2) { return dd_isqrt2() / p2; }
__device__ __forceinline__ cxd s_scale(dd f, cxd v) { return cxd_scale(f, v); }
__device__ __forceinline__ void ext_current(const double* pk, int lambda, cxd* eps) {
    dd p[4];
#pragma unroll
    for (int c = 0; c < 4; c++) p[c] = mkdd(pk[c]);
    polarisation_t<dd>(p, lambda, eps);
}
__device__ __forceinline__ dd cneg(dd v, int m) { return mkdd(cneg(v.hi, m), cneg(v.lo, m)); }
__device__ __forceinline__ cxd cneg(cxd v, int m) { return mkd(cneg(v.re, m), cneg(v.im, m)); }
__device__ __forceinline__ cxd shfl_xor(cxd v, int d) {
    return mkd(mkdd(shfl_xor(v.re.hi, d), shfl_xor(v.re.lo, d)), mkdd(shfl_xor(v.im.hi, d), shfl_xor(v.im.lo, d)));
}
__device__ __forceinline__ int hi_word(cxd v) { return __double2hiint(v.re.hi); }

cudaError_t dispatch_interp_dd(cudaStream_t s, const ProgTable* t, int sm_count, const ProgParams& p, int* launches, bool conc, bool merged,
                               long long tasks_hint) {
    if (t->dd_mode < 0 || t->dense) return cudaErrorInvalidValue;
    LaunchShape shape;
    shape.regs = 255;
    shape.conc = conc;   // small batches: the tier launches side by side, each with its share of the slabs
    shape.merged = merged;   // ... or one launch for the lists of all tiers (the capped shared state is the same for all)
    shape.cap_cx = t->dd_cap_cx;
    shape.spill_blocks = t->dd_spill_blocks;
    shape.max_blocks = t->dd_max_blocks;
    shape.tasks_hint = tasks_hint;
    // always the SPILL instantiation: offsets below the cap live in shared memory, the rest in the block's slab
    switch (t->G) {
        case 1: return launch_interp<1, true, cxd>(s, t, sm_count, p, launches, shape);
        case 2: return launch_interp<2, true, cxd>(s, t, sm_count, p, launches, shape);
        case 4: return launch_interp<4, true, cxd>(s, t, sm_count, p, launches, shape);
        case 8: return launch_interp<8, true, cxd>(s, t, sm_count, p, launches, shape);
        case 16: return launch_interp<16, true, cxd>(s, t, sm_count, p, launches, shape);
        case 32: return launch_interp<32, true, cxd>(s, t, sm_count, p, launches, shape);
        case 64: return launch_interp<64, true, cxd>(s, t, sm_count, p, launches, shape);
        case 128: return launch_interp<128, true, cxd>(s, t, sm_count, p, launches, shape);
        default: return launch_interp<256, true, cxd>(s, t, sm_count, p, launches, shape);
    }
}

}  // namespace bg
