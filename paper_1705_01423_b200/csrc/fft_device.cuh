// fft_device.cuh -- fp64 complex FFT building blocks for the periodic-direction transforms
// (paper steps 3, 5, 9, 11: P:L105-L113).  Hand-written for sm_100a; no cuFFT.
//
// A line of N complex points is transformed by NPASS Stockham (autosort, decimation in
// frequency) passes of radix R0, R1, ...  Pass p (radix R, S = R0*...*R_{p-1} interleaved
// sub-sequences, each of length L = N/S, M = L/R):
//     butterfly b = t + S*q  (t < S, q < M) reads  x[b + (N/R)*r],             r  = 0..R-1
//                                          writes y[t + S*(R*q + r')] =
//                                  w_L^{q r'} * sum_r x_r w_R^{r r'},          r' = 0..R-1
// Reads are unit-stride in b (coalesced from global memory, conflict-free from shared
// memory); the first pass takes its inputs straight from global memory / registers and the
// last pass writes straight to global memory, so a 3-pass plan makes two shared-memory
// round trips.  Only the forward transform (w = exp(-2 pi i / N)) is implemented; the
// inverse is obtained by swapping re/im on load and on store.
#pragma once
#include <cuda_runtime.h>

namespace afid {

typedef double2 cplx;

__device__ __forceinline__ cplx mk(double x, double y) { return make_double2(x, y); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return mk(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return mk(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b)
{
    return mk(fma(-a.y, b.y, a.x * b.x), fma(a.y, b.x, a.x * b.y));
}
__device__ __forceinline__ cplx cswap(cplx a) { return mk(a.y, a.x); }

// cos(2 pi k / 48) for the angles the fixed-radix butterflies need (radices 2,3,4,6,8,12,16
// only involve multiples of 2 pi / 48).  Literals are correctly rounded fp64 values.
__device__ __forceinline__ constexpr double cos48_q(int k) // 0 <= k <= 12
{
    return k == 0 ? 1.0
         : k == 1 ? 0.99144486137381041114
         : k == 2 ? 0.96592582628906828675
         : k == 3 ? 0.92387953251128675613
         : k == 4 ? 0.86602540378443864676
         : k == 5 ? 0.79335334029123516458
         : k == 6 ? 0.70710678118654752440
         : k == 7 ? 0.60876142900872063942
         : k == 8 ? 0.5
         : k == 9 ? 0.38268343236508977173
         : k == 10 ? 0.25881904510252076235
         : k == 11 ? 0.13052619222005159155
         : 0.0;
}
__device__ __forceinline__ constexpr double cos48(int k)
{
    k = ((k % 48) + 48) % 48;
    if (k > 24) k = 48 - k;
    return k > 12 ? -cos48_q(24 - k) : cos48_q(k);
}
__device__ __forceinline__ constexpr double sin48(int k) { return cos48(k - 12); }

// x * exp(-2 pi i k / 48); k folds to a constant after unrolling.
__device__ __forceinline__ cplx mul_w48(cplx x, int k)
{
    k = ((k % 48) + 48) % 48;
    if (k == 0) return x;
    if (k == 12) return mk(x.y, -x.x);
    if (k == 24) return mk(-x.x, -x.y);
    if (k == 36) return mk(-x.y, x.x);
    const double c = cos48(k), s = -sin48(k);
    return mk(fma(-x.y, s, x.x * c), fma(x.y, c, x.x * s));
}

// In-place forward DFT of R points held in registers, natural order in and out.
template <int R> struct Dft;

template <> struct Dft<1> {
    static __device__ __forceinline__ void run(cplx (&)[1]) {}
};
template <> struct Dft<2> {
    static __device__ __forceinline__ void run(cplx (&v)[2])
    {
        const cplx a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    }
};
template <> struct Dft<3> {
    static __device__ __forceinline__ void run(cplx (&v)[3])
    {
        const double hs3 = 0.86602540378443864676; // sin(pi/3)
        const cplx t1 = cadd(v[1], v[2]);
        const cplx t2 = mk(fma(-0.5, t1.x, v[0].x), fma(-0.5, t1.y, v[0].y));
        const cplx d = csub(v[1], v[2]);
        const cplx t3 = mk(hs3 * d.x, hs3 * d.y);
        v[0] = cadd(v[0], t1);
        v[1] = mk(t2.x + t3.y, t2.y - t3.x); // t2 - i t3
        v[2] = mk(t2.x - t3.y, t2.y + t3.x); // t2 + i t3
    }
};
template <> struct Dft<5> { // lengths 5 * 2^a (the paper's 1280-point direction, Table 3)
    static __device__ __forceinline__ void run(cplx (&v)[5])
    {
        const double c1 = 0.30901699437494742410, c2 = -0.80901699437494742410; // cos(2 pi/5), cos(4 pi/5)
        const double s1 = 0.95105651629515357212, s2 = 0.58778525229247312917;  // sin(2 pi/5), sin(4 pi/5)
        const cplx a1 = cadd(v[1], v[4]), a2 = cadd(v[2], v[3]), b1 = csub(v[1], v[4]), b2 = csub(v[2], v[3]);
        const cplx r1 = mk(fma(c2, a2.x, fma(c1, a1.x, v[0].x)), fma(c2, a2.y, fma(c1, a1.y, v[0].y)));
        const cplx r2 = mk(fma(c1, a2.x, fma(c2, a1.x, v[0].x)), fma(c1, a2.y, fma(c2, a1.y, v[0].y)));
        const cplx i1 = mk(fma(s2, b2.x, s1 * b1.x), fma(s2, b2.y, s1 * b1.y));
        const cplx i2 = mk(fma(-s1, b2.x, s2 * b1.x), fma(-s1, b2.y, s2 * b1.y));
        v[0] = cadd(v[0], cadd(a1, a2));
        v[1] = mk(r1.x + i1.y, r1.y - i1.x); // r1 - i i1
        v[4] = mk(r1.x - i1.y, r1.y + i1.x); // r1 + i i1
        v[2] = mk(r2.x + i2.y, r2.y - i2.x); // r2 - i i2
        v[3] = mk(r2.x - i2.y, r2.y + i2.x); // r2 + i i2
    }
};
template <> struct Dft<4> {
    static __device__ __forceinline__ void run(cplx (&v)[4])
    {
        const cplx t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        const cplx t2 = cadd(v[1], v[3]), d = csub(v[1], v[3]);
        const cplx t3 = mk(d.y, -d.x); // -i (v1 - v3)
        v[0] = cadd(t0, t2);
        v[1] = cadd(t1, t3);
        v[2] = csub(t0, t2);
        v[3] = csub(t1, t3);
    }
};

// Cooley-Tukey composite N = N1*N2 in registers:
// X[k1 + N1 k2] = sum_{n2} w_N2^{n2 k2} [ w_N^{n2 k1} sum_{n1} x[N2 n1 + n2] w_N1^{n1 k1} ]
template <int N1, int N2> struct DftCt {
    static constexpr int N = N1 * N2;
    static __device__ __forceinline__ void run(cplx (&v)[N])
    {
        cplx a[N2][N1];
#pragma unroll
        for (int n2 = 0; n2 < N2; ++n2) {
            cplx t[N1];
#pragma unroll
            for (int n1 = 0; n1 < N1; ++n1) t[n1] = v[N2 * n1 + n2];
            Dft<N1>::run(t);
#pragma unroll
            for (int k1 = 0; k1 < N1; ++k1) a[n2][k1] = mul_w48(t[k1], n2 * k1 * (48 / N));
        }
#pragma unroll
        for (int k1 = 0; k1 < N1; ++k1) {
            cplx t[N2];
#pragma unroll
            for (int n2 = 0; n2 < N2; ++n2) t[n2] = a[n2][k1];
            Dft<N2>::run(t);
#pragma unroll
            for (int k2 = 0; k2 < N2; ++k2) v[k1 + N1 * k2] = t[k2];
        }
    }
};
template <> struct Dft<6> {
    static __device__ __forceinline__ void run(cplx (&v)[6]) { DftCt<2, 3>::run(v); }
};
template <> struct Dft<8> {
    static __device__ __forceinline__ void run(cplx (&v)[8]) { DftCt<4, 2>::run(v); }
};
template <> struct Dft<12> {
    static __device__ __forceinline__ void run(cplx (&v)[12]) { DftCt<4, 3>::run(v); }
};
template <> struct Dft<16> {
    static __device__ __forceinline__ void run(cplx (&v)[16]) { DftCt<4, 4>::run(v); }
};

// A transform plan: N = R0*R1*R2*R3 (unused radices = 1), TPL threads cooperate on a line.
template <int R0_, int R1_, int R2_, int R3_, int TPL_> struct FftPlan {
    static constexpr int R0 = R0_, R1 = R1_, R2 = R2_, R3 = R3_, TPL = TPL_;
    static constexpr int N = R0 * R1 * R2 * R3;
    static constexpr int NPASS = R1 == 1 ? 1 : (R2 == 1 ? 2 : (R3 == 1 ? 3 : 4));
    // Shared-memory layout of a line: one pad element after every R0 elements, so that the
    // first pass's stride-R0 writes are bank-conflict free; line stride = 2 mod 8 (in 16-byte
    // units) so that K1's split pass, whose 8-lane phases touch slots k, k+1 of 4 lines, is too.
    static constexpr int PADDED = N + N / R0; // = pad(N): one extra slot (index N) is kept for K5's Nyquist entry
    static constexpr int LS = PADDED + ((2 - PADDED % 8) + 8) % 8 + ((PADDED % 8 == 2) ? 8 : 0); // = 2 mod 8, > PADDED
    static __device__ __forceinline__ int pad(int e) { return e + e / R0; }
    template <int P> static constexpr int radix() { return P == 0 ? R0 : (P == 1 ? R1 : (P == 2 ? R2 : R3)); }
    template <int P> static constexpr int stride() { return P == 0 ? 1 : (P == 1 ? R0 : (P == 2 ? R0 * R1 : R0 * R1 * R2)); }
};

// One pass.  ld(e) returns element e of the pass input, st(e, v) stores element e of the
// pass output; tw = table of exp(-2 pi i k / N), k < N (global memory, read-only path).
template <class PL, int P> struct FftPass {
    static constexpr int R = PL::template radix<P>();
    static constexpr int S = PL::template stride<P>();
    static constexpr int N = PL::N, TPL = PL::TPL;
    static constexpr int NB = N / R;
    static constexpr int ROUNDS = (NB + TPL - 1) / TPL;
    static constexpr int M = N / S / R;
    static constexpr bool EXACT = (NB % TPL) == 0;

    struct Regs {
        cplx v[ROUNDS][R];
    };

    template <class Load> static __device__ __forceinline__ void load(Regs& rg, int tl, Load ld)
    {
#pragma unroll
        for (int rd = 0; rd < ROUNDS; ++rd) {
            const int b = tl + rd * TPL;
            if (EXACT || b < NB) {
#pragma unroll
                for (int r = 0; r < R; ++r) rg.v[rd][r] = ld(b + NB * r);
            }
        }
    }
    template <class Store>
    static __device__ __forceinline__ void compute_store(Regs& rg, int tl, const cplx* __restrict__ tw, Store st)
    {
#pragma unroll
        for (int rd = 0; rd < ROUNDS; ++rd) {
            const int b = tl + rd * TPL;
            if (EXACT || b < NB) {
                Dft<R>::run(rg.v[rd]);
                const int t = b % S, q = b / S;
                if (M > 1) {
                    const int e = q * S;
                    if (S == 1) {
                        // first pass: every butterfly has its own twiddle base w = tw[b]; one
                        // coalesced load, the powers w^r by a depth-log2(r) product tree
                        // (a gather of tw[b*r] would touch up to 32 cache lines per warp load)
                        cplx wp[R];
                        wp[1] = __ldg(&tw[e]);
#pragma unroll
                        for (int r = 2; r < R; ++r) wp[r] = cmul(wp[r / 2], wp[r - r / 2]);
#pragma unroll
                        for (int r = 1; r < R; ++r) rg.v[rd][r] = cmul(rg.v[rd][r], wp[r]);
                    } else {
                        // later passes: S consecutive butterflies share q, the loads are broadcasts
#pragma unroll
                        for (int r = 1; r < R; ++r) rg.v[rd][r] = cmul(rg.v[rd][r], __ldg(&tw[e * r]));
                    }
                }
                const int o = t + S * R * q;
#pragma unroll
                for (int r = 0; r < R; ++r) st(o + S * r, rg.v[rd][r]);
            }
        }
    }
};

// Passes 1..NPASS-1 of a line whose pass-0 output already sits in shared memory `line`
// (padded layout); the last pass stores through `st_last`.  If LAST_TO_SMEM the last pass's
// output goes back to `line` instead (st_last unused) and a barrier follows it.
// Every thread of the CTA must call this (it contains __syncthreads()); threads with
// active == false take part in the barriers only.
// `acc(pe)` returns a reference to padded slot pe = PL::pad(e) of the line (the caller chooses where
// the slots live: a plain padded line, or a swizzled column of a TMA tile).
// `sync()` is the barrier between the passes: __syncthreads() by default; a kernel whose lines are owned by whole
// warps may pass a named barrier over just the warps of a line group (the passes of different lines are independent).
struct CtaSync {
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};
// named barrier `id` (1..15) over `nthreads` threads (a multiple of 32: whole warps)
struct GroupSync {
    int id, nthreads;
    __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }
};

struct NoHook {
    __device__ __forceinline__ void operator()() const {}
};
// `loaded()` is called once, right after the loads of the LAST pass (the line's shared-memory slots are dead from
// then on: a kernel that recycles the buffer can hand it back before the global stores).
template <class PL, int P, bool LAST_TO_SMEM, class Acc, class StoreLast, class Sync = CtaSync, class Hook = NoHook>
__device__ __forceinline__ void fft_tail_passes_acc(Acc acc, int tl, bool active, const cplx* __restrict__ tw, StoreLast st_last, Sync sync = Sync(),
                                                    Hook loaded = Hook())
{
    if constexpr (P < PL::NPASS) {
        typedef FftPass<PL, P> PS;
        typename PS::Regs rg;
        sync(); // previous pass's writes visible
        if (active) PS::load(rg, tl, [&](int e) { return acc(PL::pad(e)); });
        if constexpr (P == PL::NPASS - 1 && !LAST_TO_SMEM) {
            loaded();
            if (active) PS::compute_store(rg, tl, tw, st_last);
        } else {
            sync(); // all reads done before the in-place writes
            if (active) PS::compute_store(rg, tl, tw, [&](int e, cplx v) { acc(PL::pad(e)) = v; });
        }
        fft_tail_passes_acc<PL, P + 1, LAST_TO_SMEM>(acc, tl, active, tw, st_last, sync, loaded);
    } else {
        if constexpr (LAST_TO_SMEM) sync();
    }
}
template <class PL, int P, bool LAST_TO_SMEM, class StoreLast>
__device__ __forceinline__ void fft_tail_passes(cplx* line, int tl, bool active, const cplx* __restrict__ tw,
                                                StoreLast st_last)
{
    fft_tail_passes_acc<PL, P, LAST_TO_SMEM>([line](int pe) -> cplx& { return line[pe]; }, tl, active, tw, st_last);
}

} // namespace afid
