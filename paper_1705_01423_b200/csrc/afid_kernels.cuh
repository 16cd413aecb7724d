// afid_kernels.cuh -- the six kernels of one projection step (sm_100a, fp64).
//
//   K1 k_div_r2c     divergence (paper step 1) fused with the real-to-complex
//                    transform along z (step 3; z is our contiguous direction)
//   K2 k_fft_y       complex transform along y (step 5)
//   K3 k_solve_x     tridiagonal solve along x per (ky,kz) (step 7)
//   K4 k_ifft_y      inverse complex transform along y (step 9)
//   K5 k_c2r_z       inverse complex-to-real transform along z (step 11) -> p = phi
//   K6 k_correct     velocity correction u -= G phi
//
// The paper's pencil transposes (steps 2,4,6,8,10,12) become the tile gathers of K2..K5:
// every kernel writes its output contiguously and the NEXT kernel gathers >=128-byte
// segments (measured on B200: segmented reads of >=256 B run at copy speed, segmented
// writes do not).  Work-array layouts (complex doubles; nzh = nz/2+1, NJT = ny/8):
//   B  [i][jt][kz][8]     written by K1   (8 = j within the tile jt)
//   C  [kz][i][ky]        written by K2   (kz-major: the rows i of a K3 tile are ny*16 bytes apart, not a plane apart)
//   T  [kz][kyt][i][8]    written by K3   (8 = ky within the tile kyt)
//   D  [i][kz][j]         written by K4
#pragma once
#include "fft_device.cuh"
#include "tma.cuh"

namespace afid {

struct DevParams {
    int nx, ny, nz, nzh;
    double rdy, rdz;            // 1/dy, 1/dz
    double spec_scale;          // -1/(ny*nz): folded into K1's post-processing
    const double* rdx;          // [nx]   1/dx_i
    const double* rdc;          // [nx+1] 1/dc_i (faces 1..nx-1; 0 at the walls)
    const double* dxw;          // [nx]   dx_i (weights of the mean)
    const double* ca;           // [nx]   a_i = 1/(dx_i dc_i),   a_0 = 0
    const double* cc;           // [nx]   c_i = 1/(dx_i dc_{i+1}), c_{nx-1} = 0
    const double2* acp;         // K3: {a_i, c_i} in the kernel's shared-memory layout (chunk q at [q (M+1), q (M+1) + M]), k3_coef_slots entries
    const double* lamy;         // [ny]   modified wavenumbers in y
    const double* lamz;         // [nzh]  modified wavenumbers in z
    const cplx* tw_y;           // [ny]    exp(-2 pi i k/ny)
    const cplx* tw_zh;          // [nz/2]  exp(-2 pi i k/(nz/2))
    const cplx* tw_z;           // [nz/2+1] exp(-2 pi i k/nz)
    double inv_vol;             // 1/sum dx_i
    int hints;                  // L2 eviction-priority switches (bit mask, see l2_policy users)
    int k3_prefetch;            // K3: a CTA prefetches the tile of CTA blockIdx.x + k3_prefetch into L2 (0 = off)
    int has_mean;               // K3: this launch holds the mean mode (ky, kz) = (0, 0) as its first system (sharded plans: only the rank owning kz = 0)
};

// L2 eviction priorities (PTX createpolicy): 0 = normal, 1 = evict_first (streamed once), 2 = evict_last (kept)
__device__ __forceinline__ unsigned long long l2_policy(int kind)
{
    unsigned long long p;
    if (kind == 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    else if (kind == 2) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ double2 ldv2h(const double* p, unsigned long long pol)
{
    double2 r;
    asm volatile("ld.global.nc.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(r.x), "=d"(r.y) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ double ldv1h(const double* p, unsigned long long pol)
{
    double r;
    asm volatile("ld.global.nc.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(r) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ cplx ldc_h(const cplx* p, unsigned long long pol)
{
    cplx r;
    asm volatile("ld.global.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(r.x), "=d"(r.y) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ void stc_h(cplx* p, cplx v, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}

__device__ __forceinline__ double2 ldg2(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }
// a register "pin": see K1
// scheduling fence between a load batch and its consumers; only the converged lanes take part
// (the callers sit inside `if (act)`: a full-mask __syncwarp there would hang on partial warps)
#define SCHED_FENCE() __syncwarp(__activemask())
__device__ __forceinline__ void pin(double2& a) { asm volatile("" : "+d"(a.x), "+d"(a.y)); }
__device__ __forceinline__ void pin1(double& a) { asm volatile("" : "+d"(a)); }

// ------------------------------------------------------------------------------------------
// K1: divergence + r2c along z.  CTA = (i, group of NL consecutive j); NL*TPL threads.
// The real line d(i,j,0..nz-1) is transformed as the complex line z(m) = d(2m) + i d(2m+1)
// of length Nh = nz/2, then split:  X(k) = 1/2 [ (Z(k)+conj Z(Nh-k)) - i w_nz^k (Z(k)-conj Z(Nh-k)) ].
// Output: B[i][jt][kz][jl] = spec_scale * X(kz), kz = 0..Nh.
// ------------------------------------------------------------------------------------------
template <class PL, int NL>
__global__ void __launch_bounds__(NL* PL::TPL, (NL * PL::TPL <= 256) ? 2 : 1) k_div_r2c(DevParams P, const double* __restrict__ u,
                                                         const double* __restrict__ v, const double* __restrict__ w,
                                                         cplx* __restrict__ B, int i_base, int np, int bmod)
{
    constexpr int Nh = PL::N, TPL = PL::TPL, LS = PL::LS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* sm = reinterpret_cast<cplx*>(smem_raw);
    // CTA order: j-chunks of JC groups outermost, then i, then the group inside the chunk, so
    // that plane i+1 of u (read again as plane i of the next step in i) is still in L2
    const int ngrp = P.ny / NL;
    constexpr int JC = 64 / NL;
    // this launch covers planes i_base .. i_base+np-1
    const int per_chunk = np * JC;
    int i, jg;
    {
        const int chunk = blockIdx.x / per_chunk, rem = blockIdx.x % per_chunk;
        const int jc_here = min(JC, ngrp - chunk * JC);
        i = i_base + rem / jc_here;
        jg = chunk * JC + rem % jc_here;
    }
    const size_t plane = (size_t)P.ny * P.nz;
    const int ln = threadIdx.x / TPL, tl = threadIdx.x % TPL;
    const int j = jg * NL + ln;
    const int jp = (j + 1 == P.ny) ? 0 : j + 1;
    const double* u0 = u + (size_t)i * plane + (size_t)j * P.nz;
    const double* u1 = u0 + plane;
    const double* v0 = v + (size_t)i * plane + (size_t)j * P.nz;
    const double* v1 = v + (size_t)i * plane + (size_t)jp * P.nz;
    const double* w0 = w + (size_t)i * plane + (size_t)j * P.nz;
    const double rdx = __ldg(&P.rdx[i]), rdy = P.rdy, rdz = P.rdz;
    cplx* line = sm + ln * LS;
    const unsigned long long pol_in = l2_policy((P.hints & 1) ? 1 : 0), pol_u1 = l2_policy(0);
    const unsigned long long pol_b = l2_policy((P.hints & 2) ? 2 : 0);

    // divergence of the two cells 2e, 2e+1 (P:L87 stencil).  The loads are issued in batches
    // of 2*NBATCH independent 16-byte loads (volatile PTX keeps them together; `pin` makes the
    // arithmetic wait for the whole batch) -- otherwise ptxas interleaves each load with its
    // consumer and the kernel is latency-bound at 2-3 loads in flight per thread.
    {
        typedef FftPass<PL, 0> P0;
        constexpr int R = P0::R, NB = P0::NB;
        // one batch = all five streams of NBATCH element pairs: 5 NBATCH 16-byte loads + NBATCH 8-byte loads in flight per
        // thread, R / NBATCH round trips to memory per CTA (separate u, v, w batches of 8 loads needed 12 round trips for
        // R = 16; ncu: the load phase is 46 % of the kernel, all of it long-scoreboard stalls at 12 warps per SM)
        constexpr int NBATCH = (R % 2 == 0) ? 2 : 1;
        static_assert(P0::ROUNDS == 1, "K1 expects one first-pass butterfly per thread");
        typename P0::Regs rg;
        const bool act = P0::EXACT || tl < NB;
        if (act) {
#pragma unroll
            for (int h = 0; h < R; h += NBATCH) {
                double2 a1[NBATCH], a0[NBATCH], b1[NBATCH], b0[NBATCH], c0[NBATCH];
                double cn[NBATCH];
#pragma unroll
                for (int r = 0; r < NBATCH; ++r) {
                    const int e = tl + NB * (h + r);
                    a1[r] = ldv2h(u1 + 2 * e, pol_u1);
                    a0[r] = ldv2h(u0 + 2 * e, pol_in);
                    b1[r] = ldv2h(v1 + 2 * e, pol_u1);
                    b0[r] = ldv2h(v0 + 2 * e, pol_in);
                    c0[r] = ldv2h(w0 + 2 * e, pol_in);
                    cn[r] = ldv1h(w0 + ((e == Nh - 1) ? 0 : 2 * e + 2), pol_in);
                }
                SCHED_FENCE();
#pragma unroll
                for (int r = 0; r < NBATCH; ++r) { pin(a1[r]); pin(a0[r]); pin(b1[r]); pin(b0[r]); pin(c0[r]); pin1(cn[r]); }
#pragma unroll
                for (int r = 0; r < NBATCH; ++r) {
                    double dx_ = (a1[r].x - a0[r].x) * rdx, dy_ = (a1[r].y - a0[r].y) * rdx;
                    dx_ = fma(b1[r].x - b0[r].x, rdy, dx_);
                    dy_ = fma(b1[r].y - b0[r].y, rdy, dy_);
                    dx_ = fma(c0[r].y - c0[r].x, rdz, dx_);
                    dy_ = fma(cn[r] - c0[r].y, rdz, dy_);
                    rg.v[0][h + r] = mk(dx_, dy_);
                }
            }
            P0::compute_store(rg, tl, P.tw_zh, [&](int e, cplx val) { line[PL::pad(e)] = val; });
        }
    }
    constexpr int SPLIT_N = (Nh / 2 + 1) * NL;
    {   // barriers between the passes only over the warps of a line group (see K5); the split below needs all lines
        constexpr int GL = (TPL % 32 == 0) ? 1 : ((2 * TPL) % 32 == 0 ? 2 : 4);
        if constexpr (GL < NL && (GL * TPL) % 32 == 0) {
            const GroupSync gsync{1 + ln / GL, GL * TPL};
            fft_tail_passes_acc<PL, 1, true>([line](int pe) -> cplx& { return line[pe]; }, tl, true, P.tw_zh, [](int, cplx) {}, gsync);
            __syncthreads();
        } else {
            fft_tail_passes<PL, 1, true>(line, tl, true, P.tw_zh, [](int, cplx) {});
        }
    }

    // split into the spectrum of the real line; thread -> (k, jl) with jl fastest
    const int jl0 = (jg * NL) % 8;         // position of this CTA's first line inside the tile
    // B may be a rotating buffer of bmod planes (plane-batched launches keep it L2-resident)
    cplx* out = B + ((size_t)(i % bmod) * (P.ny / 8) + (size_t)(jg * NL / 8)) * (size_t)P.nzh * 8;
    const double hs = 0.5 * P.spec_scale;
    // the twiddle of the NEXT iteration is always in flight (ncu: the load -> use latency inside this loop was 7 % of
    // the kernel's stall samples)
    cplx wk_next = __ldg(&P.tw_z[min((int)threadIdx.x, SPLIT_N - 1) / NL]);
    for (int idx = threadIdx.x; idx < SPLIT_N; idx += NL * TPL) {
        const int k = idx / NL, l = idx % NL;
        const cplx* zl = sm + l * LS;
        const cplx zk = zl[PL::pad(k)];
        const cplx zm = zl[PL::pad(k == 0 ? 0 : Nh - k)];
        // E = Z(k) + conj Z(Nh-k);  O = Z(k) - conj Z(Nh-k)
        const cplx E = mk(zk.x + zm.x, zk.y - zm.y), O = mk(zk.x - zm.x, zk.y + zm.y);
        const cplx wk = wk_next; // exp(-2 pi i k / nz)
        if (idx + NL * TPL < SPLIT_N) wk_next = __ldg(&P.tw_z[(idx + NL * TPL) / NL]);
        // -i w O
        const cplx wo = cmul(wk, O);
        const cplx t = mk(wo.y, -wo.x);
        const cplx xk = mk(hs * (E.x + t.x), hs * (E.y + t.y));
        // X(Nh-k) = 1/2 [ conj(E) ... ]: by symmetry X(Nh-k) = 1/2 conj( E + i w O ) ... derived below
        // Z(Nh-k) + conj Z(k) = conj(E);  Z(Nh-k) - conj Z(k) = -conj(O);  w^(Nh-k) = -conj(w^k)
        // X(Nh-k) = 1/2 [ conj(E) - i (-conj w)(-conj O) ] = 1/2 [ conj(E) - i conj(w O) ] = 1/2 conj( E + i w O )
        const cplx xm = mk(hs * (E.x - t.x), -hs * (E.y - t.y));
        stc_h(&out[(size_t)k * 8 + jl0 + l], xk, pol_b);
        if (k != Nh - k) stc_h(&out[(size_t)(Nh - k) * 8 + jl0 + l], xm, pol_b);
    }
}

// ------------------------------------------------------------------------------------------
// K2: forward complex FFT along y.  CTA = (i, NL consecutive kz); reads B (segments of
// NL*128 bytes), writes C[kz][i][ky] contiguously.
// ------------------------------------------------------------------------------------------
template <class PL> constexpr int tpl8() { return (PL::TPL + 7) / 8 * 8; }

template <class PL, int NL>
__global__ void __launch_bounds__(NL* tpl8<PL>(), (NL * tpl8<PL>() <= 192) ? 3 : ((NL * tpl8<PL>() <= 256) ? 2 : 1)) k_fft_y(DevParams P, const cplx* __restrict__ B, cplx* __restrict__ C, int i_base, int bmod)
{
    constexpr int TPL = PL::TPL, LS = PL::LS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* sm = reinterpret_cast<cplx*>(smem_raw);
    const int ngrp = (P.nzh + NL - 1) / NL;
    const int i = i_base + blockIdx.x / ngrp, kg = blockIdx.x % ngrp;
    // interleave the NL lines at 8-thread granularity so that a warp's loads cover
    // NL*128 contiguous bytes of B
    const int ln = (threadIdx.x >> 3) % NL;
    const int tl = (threadIdx.x & 7) | ((threadIdx.x / (8 * NL)) << 3);
    const int kz = kg * NL + ln;
    const bool active = (kz < P.nzh) && (tl < TPL);
    const cplx* src = B + (size_t)(i % bmod) * (P.ny / 8) * (size_t)P.nzh * 8 + (size_t)kz * 8;
    const size_t tile_stride = (size_t)P.nzh * 8;
    cplx* dst = C + ((size_t)kz * P.nx + i) * (size_t)P.ny;
    cplx* line = sm + ln * LS;
    const unsigned long long pol_b = l2_policy((P.hints & 4) ? 1 : ((P.hints & 2) ? 2 : 0));
    const unsigned long long pol_c = l2_policy((P.hints & 8) ? 1 : 0);
    auto ld_b = [&](int e) -> cplx {
        const cplx* a = &src[(size_t)(e >> 3) * tile_stride + (e & 7)];
        const cplx r = ldc_h(a, pol_b);
        return r;
    };
    auto st_c = [&](int e, cplx val) { stc_h(&dst[e], val, pol_c); };
    typedef FftPass<PL, 0> P0;
    if constexpr (PL::NPASS == 1) {
        if (active) {
            typename P0::Regs rg;
            P0::load(rg, tl, ld_b);
            P0::compute_store(rg, tl, P.tw_y, st_c);
        }
    } else {
        if (active) {
            typename P0::Regs rg;
            P0::load(rg, tl, ld_b);
            P0::compute_store(rg, tl, P.tw_y, [&](int e, cplx val) { line[PL::pad(e)] = val; });
        }
        fft_tail_passes<PL, 1, false>(line, tl, active, P.tw_y, st_c);
    }
}

// ------------------------------------------------------------------------------------------
// K4: inverse complex FFT along y (unnormalised; the 1/(ny nz) is in spec_scale).
// CTA = (NL consecutive i, kz); reads T[kz][kyt][i][8] (segments of NL*128 bytes), writes
// D[i][kz][j] contiguously.  Inverse = forward with re/im swapped on load and store.
// ------------------------------------------------------------------------------------------
template <class PL, int NL>
__global__ void __launch_bounds__(NL* tpl8<PL>(), (NL * tpl8<PL>() <= 192) ? 3 : ((NL * tpl8<PL>() <= 256) ? 2 : 1)) k_ifft_y(DevParams P, const cplx* __restrict__ T, cplx* __restrict__ D, int i_base, int np,
                                                         int dmod)
{
    constexpr int TPL = PL::TPL, LS = PL::LS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx* sm = reinterpret_cast<cplx*>(smem_raw);
    // this launch covers planes i_base .. i_base+np-1; D may be a rotating buffer of dmod planes
    const int ngrp = (np + NL - 1) / NL;
    const int kz = blockIdx.x / ngrp, ig = blockIdx.x % ngrp;
    const int ln = (threadIdx.x >> 3) % NL;
    const int tl = (threadIdx.x & 7) | ((threadIdx.x / (8 * NL)) << 3);
    const int i = i_base + ig * NL + ln;
    const bool active = (i < i_base + np) && (tl < TPL);
    const size_t tile_stride = (size_t)P.nx * 8;
    const cplx* src = T + (size_t)kz * (P.ny / 8) * tile_stride + (size_t)i * 8;
    cplx* dst = D + ((size_t)(i % dmod) * P.nzh + kz) * (size_t)P.ny;
    cplx* line = sm + ln * LS;
    const unsigned long long pol_t = l2_policy((P.hints & 1) ? 1 : 0), pol_d = l2_policy((P.hints & 2) ? 2 : 0);
    auto ld_t = [&](int e) -> cplx { return cswap(ldc_h(&src[(size_t)(e >> 3) * tile_stride + (e & 7)], pol_t)); };
    auto st_d = [&](int e, cplx val) { stc_h(&dst[e], cswap(val), pol_d); };
    typedef FftPass<PL, 0> P0;
    if constexpr (PL::NPASS == 1) {
        if (active) {
            typename P0::Regs rg;
            P0::load(rg, tl, ld_t);
            P0::compute_store(rg, tl, P.tw_y, st_d);
        }
    } else {
        if (active) {
            typename P0::Regs rg;
            P0::load(rg, tl, ld_t);
            P0::compute_store(rg, tl, P.tw_y, [&](int e, cplx val) { line[PL::pad(e)] = val; });
        }
        fft_tail_passes<PL, 1, false>(line, tl, active, P.tw_y, st_d);
    }
}

// ------------------------------------------------------------------------------------------
// K5: inverse c2r along z -> p.  CTA = (i, tile of 8 consecutive j); LPR*TPL threads process the
// 8 lines in 8/LPR rounds of LPR lines (registers hold one round; two CTAs per SM overlap one
// CTA's gather with the other's transform).
// Gathers D[i][kz][8 j] (128-byte segments, cp.async), forms in place
//   Z'(k) = (X(k)+conj X(Nh-k)) + i conj(w^k)(X(k)-conj X(Nh-k)),
// inverse complex FFT of length Nh gives z(m) = phi(2m) + i phi(2m+1).
// ------------------------------------------------------------------------------------------
// TMA tile of K5: (Nh+1) rows kz of 128 bytes (8 j), fetched as k5_num_boxes boxes of k5_box_rows rows
// (a multiple of 8, so that every box starts on a 1024-byte swizzle period); rows >= nz/2+1 are out of
// bounds and arrive as zeros.  The shared-memory tile also has to hold the padded rows of the FFT passes.
__host__ __device__ constexpr int k5_num_boxes(int nh) { return (nh + 1 + 255) / 256; }
__host__ __device__ constexpr int k5_box_rows(int nh) { return ((nh + 1 + k5_num_boxes(nh) - 1) / k5_num_boxes(nh) + 7) / 8 * 8; }
template <class PL> constexpr int k5_smem_rows()
{
    constexpr int tma_rows = k5_num_boxes(PL::N) * k5_box_rows(PL::N);
    constexpr int fft_rows = (PL::PADDED + 8) / 8 * 8;
    return tma_rows > fft_rows ? tma_rows : fft_rows;
}

// Persistent: the launch has (at most) one CTA per SM (two for NBUF = 1), each walks over the tiles
// t = blockIdx.x, blockIdx.x + gridDim.x, ... of planes i_base .. i_base+np-1.  With NBUF = 2 the tile of the next
// step is gathered by TMA into the other buffer while this one is transformed, so HBM always has a request of
// this SM in flight (the non-persistent version waited for its whole tile before doing anything: 17 % of its
// stall samples).  A buffer is handed back to the async proxy (TMA writes) after a proxy fence and a CTA barrier.
// STW: the pre-processing twiddles exp(-2 pi i k / nz) are staged in shared memory (wherever they fit beside the tiles)
template <class PL, int LPR, int NBUF, bool STW>
__global__ void __launch_bounds__(LPR* PL::TPL, 1) k_c2r_z(DevParams P, const __grid_constant__ CUtensorMap mapD, double* __restrict__ p, int i_base, int np,
                                                           int dmod)
{
    constexpr int Nh = PL::N, TPL = PL::TPL, NL = 8, NT = LPR * TPL;
    constexpr int TILE = k5_smem_rows<PL>() * 8;     // complex slots per buffer
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar[NBUF];      // "full": the TMA gather of a buffer has landed
    __shared__ __align__(8) uint64_t empty[NBUF];    // "empty": every thread is done with the buffer's shared memory
    // 1024-byte aligned tiles [row][8 chunks of 16 bytes]; line l, row r lives in chunk l ^ (r & 7)
    // (the 128-byte TMA swizzle, kept for the in-place FFT passes: conflict-free for unit-stride rows)
    cplx* sm0 = reinterpret_cast<cplx*>(smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u)); // (offset form keeps the shared state space)
    cplx* stw = sm0 + (size_t)NBUF * TILE;           // exp(-2 pi i k / nz), k = 0..Nh: the pre-processing twiddles (ncu: their global loads
                                                     // were 6 % of the stall samples; the persistent CTA stages them once)
    const int njt = P.ny / 8;
    const int ntile = np * njt;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int b = 0; b < NBUF; ++b) { mbar_init(&bar[b], 1); mbar_init(&empty[b], NT); }
        fence_mbar_init();
    }
    if constexpr (STW)
        for (int k = threadIdx.x; k <= Nh; k += NT) stw[k] = __ldg(&P.tw_z[k]);
    __syncthreads();
    const unsigned long long pol = l2_policy((P.hints & 4) ? 1 : ((P.hints & 2) ? 2 : 0));
    auto issue = [&](int t, int buf) {   // one thread: gather tile t into buffer buf
        constexpr int nb = k5_num_boxes(Nh), br = k5_box_rows(Nh);
        const int i = i_base + t / njt, jt = t % njt;
        mbar_expect_tx(&bar[buf], (uint32_t)(nb * br * 8 * sizeof(cplx)));
        for (int b = 0; b < nb; ++b) tma_load_3d_hint(sm0 + (size_t)buf * TILE + (size_t)b * br * 8, &mapD, jt * 16, b * br, i % dmod, &bar[buf], pol);
    };
    if (threadIdx.x == 0 && (int)blockIdx.x < ntile) issue(blockIdx.x, 0);
    const int lr = threadIdx.x / TPL, tl = threadIdx.x % TPL;
    // The passes of different lines are independent: the barriers between them only span the warps of a line
    // group (the fewest lines that fill whole warps), so that one group's barrier wait is another group's issue slot.
    constexpr int GL = (TPL % 32 == 0) ? 1 : ((2 * TPL) % 32 == 0 ? 2 : ((4 * TPL) % 32 == 0 ? 4 : 8));   // lines per group
    constexpr bool GROUPED = (GL < LPR) && (LPR / GL <= 8);
    const GroupSync gsync{1 + lr / GL, GROUPED ? GL * TPL : LPR * TPL};
    auto sync = [&]() {
        if constexpr (GROUPED) gsync();
        else __syncthreads();
    };
    int n = 0;
#pragma unroll 1
    for (int t = blockIdx.x; t < ntile; t += gridDim.x, ++n) {
        const int buf = (NBUF == 2) ? (n & 1) : 0;
        if (NBUF == 2 && threadIdx.x == 0 && t + (int)gridDim.x < ntile) {
            // the other buffer held the tile of step n-1: wait until all threads have handed it back (its use number (n-1)/2)
            if (n >= 1) mbar_wait(&empty[buf ^ 1], (uint32_t)(((n - 1) >> 1) & 1));
            issue(t + gridDim.x, buf ^ 1);
        }
        cplx* sm = sm0 + (size_t)buf * TILE;
        const int i = i_base + t / njt, jt = t % njt;
        auto at = [sm](int l, int r) -> cplx& { return sm[(r << 3) + (l ^ (r & 7))]; };
        mbar_wait(&bar[buf], (NBUF == 2) ? ((n >> 1) & 1) : (n & 1));
        // Hermitian pre-processing fused into the first pass's loads: element e of the complex line is
        //   Z'(e) = (X(e) + conj X(Nh-e)) + i conj(w^e) (X(e) - conj X(Nh-e)),   w = exp(-2 pi i / nz),
        // formed from rows k = min(e, Nh-e) and Nh-k (stored re/im-swapped: the inverse runs as a forward transform)
        auto zprime = [&](int l, int e) -> cplx {
            const int k = min(e, Nh - e), km = Nh - k;
            const cplx xk = at(l, k);
            const cplx xm = at(l, km);
            const cplx wk = STW ? stw[k] : __ldg(&P.tw_z[k]);
            const cplx E = mk(xk.x + xm.x, xk.y - xm.y), O = mk(xk.x - xm.x, xk.y + xm.y);
            const cplx wo = mk(fma(wk.y, O.y, wk.x * O.x), fma(-wk.y, O.x, wk.x * O.y)); // conj(w) * O
            const cplx tt = mk(-wo.y, wo.x);                                             // i conj(w) O
            return (e == k) ? mk(E.y + tt.y, E.x + tt.x) : mk(-(E.y - tt.y), E.x - tt.x);
        };
#pragma unroll 1
        for (int rnd = 0; rnd < NL / LPR; ++rnd) {
            const int ln = rnd * LPR + lr;
            const bool last_round = (rnd == NL / LPR - 1);
            double* dst = p + ((size_t)i * P.ny + (size_t)jt * 8 + ln) * (size_t)P.nz;
            auto st_p = [&](int e, cplx val) { reinterpret_cast<double2*>(dst)[e] = cswap(val); };
            auto acc = [sm, ln](int pe) -> cplx& { return sm[(pe << 3) + (ln ^ (pe & 7))]; };
            // after the last shared-memory read of the tile (before the global stores of p): hand the buffer back to the
            // TMA (async proxy).  Only the issuing thread ever waits for it (at the top of the next step), so nobody
            // stalls on the stores (ncu: the fence + CTA barrier after the stores were 11 % of the stall samples).
            auto release = [&]() {
                if (NBUF == 2 && last_round) {
                    fence_proxy_async();
                    mbar_arrive(&empty[buf]);
                }
            };
            typedef FftPass<PL, 0> P0;
            {
                typename P0::Regs rg;
                P0::load(rg, tl, [&](int e) { return zprime(ln, e); });   // unpadded rows, as TMA delivered them
                if constexpr (PL::NPASS == 1) {
                    release();
                    P0::compute_store(rg, tl, P.tw_zh, st_p);
                } else {
                    sync();
                    P0::compute_store(rg, tl, P.tw_zh, [&](int e, cplx val) { acc(PL::pad(e)) = val; });
                }
            }
            if constexpr (PL::NPASS > 1) fft_tail_passes_acc<PL, 1, false>(acc, tl, true, P.tw_zh, st_p, sync, release);
        }
        if (NBUF == 1) {   // one buffer: it goes back to the TMA once every thread has passed this point
            fence_proxy_async();
            __syncthreads();
            if (threadIdx.x == 0 && t + (int)gridDim.x < ntile) issue(t + gridDim.x, 0);
        }
    }
}

// ------------------------------------------------------------------------------------------
// K6: correction.  CTA = (i, JL consecutive lines j); thread (x, y): line y, cell pairs
// (2k, 2k+1) for k = x, x+TX, ... in batches of U pairs (all loads of a batch issued first).
//   u[i] -= (phi[i]-phi[i-1])/dc_i (i >= 1; wall planes untouched), v -= d_y phi/dy, w -= d_z phi/dz.
// ------------------------------------------------------------------------------------------
constexpr int K6_JL = 4, K6_TX = 64, K6_U = 4;

// the correction of the lines (i, JL jg .. JL jg + JL - 1); called by all K6_JL x K6_TX threads of a CTA
// (U = cell pairs per thread and load batch)
template <int U>
__device__ __forceinline__ void k6_correct_item(const DevParams& P, const double* __restrict__ p, double* __restrict__ u, double* __restrict__ v,
                                                double* __restrict__ w, int i, int jg, double* __restrict__ pacc, const double* __restrict__ p_halo,
                                                unsigned long long pol_in, unsigned long long pol_out)
{
    constexpr int JL = K6_JL, TX = K6_TX;
    const int j = jg * JL + threadIdx.y;
    const int jm = (j == 0) ? P.ny - 1 : j - 1;
    const size_t plane = (size_t)P.ny * P.nz;
    const size_t ol = ((size_t)i * P.ny + j) * P.nz;
    const double* pl = p + ol;
    const double* pjm = p + ((size_t)i * P.ny + jm) * P.nz;
    const double* pim = (i >= 1) ? pl - plane : p_halo + (size_t)j * P.nz;   // only dereferenced if has_u
    double *ul = u + ol, *vl = v + ol, *wl = w + ol;
    const int nzh2 = P.nz / 2;
    const bool has_u = (i >= 1) || (p_halo != nullptr);
    const double rdc = has_u ? __ldg(&P.rdc[i]) : 0.0, rdy = P.rdy, rdz = P.rdz;
    for (int k0 = threadIdx.x; k0 < nzh2; k0 += TX * U) {
        double2 ph[U], pj[U], pi[U], uu[U], vv[U], ww[U];
        double pk[U];
#pragma unroll
        for (int r = 0; r < U; ++r) {
            const int kp = k0 + r * TX;
            if (kp < nzh2) {
                ph[r] = ldg2(pl + 2 * kp);
                pj[r] = ldg2(pjm + 2 * kp);
                pk[r] = __ldg(pl + (kp == 0 ? P.nz - 1 : 2 * kp - 1));
                vv[r] = ldc_h(reinterpret_cast<const cplx*>(vl + 2 * kp), pol_in);
                ww[r] = ldc_h(reinterpret_cast<const cplx*>(wl + 2 * kp), pol_in);
                if (has_u) {
                    pi[r] = ldg2(pim + 2 * kp);
                    uu[r] = ldc_h(reinterpret_cast<const cplx*>(ul + 2 * kp), pol_in);
                }
            }
        }
#pragma unroll
        for (int r = 0; r < U; ++r) {
            const int kp = k0 + r * TX;
            if (kp < nzh2) {
                vv[r].x -= (ph[r].x - pj[r].x) * rdy;
                vv[r].y -= (ph[r].y - pj[r].y) * rdy;
                ww[r].x -= (ph[r].x - pk[r]) * rdz;
                ww[r].y -= (ph[r].y - ph[r].x) * rdz;
                stc_h(reinterpret_cast<cplx*>(vl + 2 * kp), vv[r], pol_out);
                stc_h(reinterpret_cast<cplx*>(wl + 2 * kp), ww[r], pol_out);
                if (pacc) {
                    double2* q = reinterpret_cast<double2*>(pacc + ol + 2 * kp);
                    double2 t = *q;
                    t.x += ph[r].x;
                    t.y += ph[r].y;
                    *q = t;
                }
                if (has_u) {
                    uu[r].x -= (ph[r].x - pi[r].x) * rdc;
                    uu[r].y -= (ph[r].y - pi[r].y) * rdc;
                    stc_h(reinterpret_cast<cplx*>(ul + 2 * kp), uu[r], pol_out);
                }
            }
        }
    }
}

// item s of the CTA order of K6 -> (plane i, line group jg): j-chunks of JC groups outermost, then i, then the group inside
// the chunk, so that plane i-1 of p (read again for the x-gradient) is still in L2 when plane i is processed
constexpr int K6_JC = 32 / K6_JL;
__host__ __device__ __forceinline__ void k6_item_to_ij(int s, int np, int ngrp, int& i, int& jg)
{
    const int per_chunk = np * K6_JC;
    const int chunk = s / per_chunk, rem = s % per_chunk;
    const int jc_here = (K6_JC < ngrp - chunk * K6_JC) ? K6_JC : ngrp - chunk * K6_JC;
    i = rem / jc_here;
    jg = chunk * K6_JC + rem % jc_here;
}
__host__ __device__ __forceinline__ int k6_ij_to_item(int i, int jg, int np, int ngrp)
{
    const int chunk = jg / K6_JC;
    const int jc_here = (K6_JC < ngrp - chunk * K6_JC) ? K6_JC : ngrp - chunk * K6_JC;
    return chunk * np * K6_JC + i * jc_here + (jg - chunk * K6_JC);
}

__global__ void __launch_bounds__(K6_JL* K6_TX) k_correct(DevParams P, const double* __restrict__ p, double* __restrict__ u,
                                                          double* __restrict__ v, double* __restrict__ w, int i_base, int np, double* __restrict__ pacc,
                                                          const double* __restrict__ p_halo)
{
    // `p` holds phi; if pacc != nullptr the pressure is accumulated as well: pacc += phi (P:L91, P:L116 delta form).
    // p_halo (sharded plans): the plane of phi below this slab's first plane (nullptr: plane 0 is the wall)
    // this launch covers planes i_base .. i_base+np-1.
    int i, jg;
    k6_item_to_ij((int)blockIdx.x, np, P.ny / K6_JL, i, jg);
    k6_correct_item<K6_U>(P, p, u, v, w, i_base + i, jg, pacc, p_halo, l2_policy((P.hints & 1) ? 1 : 0), l2_policy((P.hints & 8) ? 1 : 0));
}

// ------------------------------------------------------------------------------------------
// K3: tridiagonal solves along x (paper step 7).  For every mode (ky,kz), lam = lamy+lamz:
//     -a_i x_{i-1} + (a_i + c_i + lam) x_i - c_i x_{i+1} = f_i ,   f = -dhat/(ny nz)  (from K1)
// (the paper's system a x_{i-1} - (a+c+lam) x_i + c x_{i+1} = dhat with the sign flipped so
// that the matrix is an M-matrix).  CTA = 8 consecutive ky of one kz; the 8 whole columns
// (nx x 8 complex) sit in shared memory; thread (s, q) owns the chunk of M rows q of system s.
//
// Parallel-in-x algorithm, every quantity a sum/product of non-negative numbers (no
// cancellation at small lam):
//   chunk q = rows [qM, qM+M); its last row is an INTERFACE unknown E_q, the others are interior.
//   1. downward elimination of the interior (one reciprocal per row):  x_i = y_i + g_i x_{i+1} + h_i E_{q-1}
//        nh = a h', nt = lam + a t', pi = c + nh + nt, h = nh/pi, t = nt/pi, g = c/pi, y = (f + a y')/pi   (g + h + t = 1)
//   2. in the same sweep, by prefix products Pg = g_0 ... g_{r-1}: the chunk's FIRST interior row in terms of
//      both interfaces,  x_{i0} = Y + Gq E_q + Hq E_{q-1},   Y = sum Pg y_r, Hq = sum Pg h_r, Gq = prod g,
//      Tq = 1 - Gq - Hq = sum Pg t_r  (a sum of non-negatives)
//   -> reduced system in E of the same form: -A_q E_{q-1} + (A_q + C_q + L_q) E_q - C_q E_{q+1} = F_q
//        A_q = a h, L_q = lam + a t + c Tq^, F_q = f + a y + c Y^, C_q = c Gq^   (^ = chunk q+1's first-row relation)
//   -> solved by cancellation-free parallel cyclic reduction across the chunks of a system
//      (L' = L + alpha L_- + gamma L_+ stays a sum of non-negatives)
//   -> interior rows by back substitution x_i = y_i + g_i x_{i+1} + h_i E_{q-1}.
// Mode (0,0) (lam = 0, singular; R7): last row pinned to 0, then the dx-weighted
// mean is subtracted.
// ------------------------------------------------------------------------------------------
// 1/x for a positive, normal x, to fp64 round-off.  The 64-bit MUFU (rcp.approx.f64, MUFU.RCP64H) is
// what the x-solve was bound by on B200 (XU pipe at 160 % of its sustained peak in ncu), so the seed is a
// 32-bit MUFU.RCP of the mantissa, moved between the formats with integer operations only (no F2F
// conversions: they use the same slow pipe), followed by ONE third-order step: with e = 1 - x r0, |e| <= 2^-22,
// r = r0 (1 + e + e^2) has relative error e^3 = 2^-66 (three dependent FMAs; two Newton steps need four).
__device__ __forceinline__ double fast_rcp(double x)
{
    const int hi = __double2hiint(x), lo = __double2loint(x);
    const unsigned fb = 0x3F800000u | ((unsigned)(hi & 0xFFFFF) << 3) | ((unsigned)lo >> 29); // 1.m as a float in [1, 2)
    float rf;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rf) : "f"(__uint_as_float(fb)));                 // in (0.5, 1]
    const unsigned rb = __float_as_uint(rf);
    const int ex = (hi >> 20) & 0x7FF;
    const int rexp = (int)(rb >> 23) + (1023 - 127) - (ex - 1023);
    const double r = __hiloint2double((rexp << 20) | (int)((rb >> 3) & 0xFFFFF), (int)(rb << 29));
    const double e = fma(-x, r, 1.0);
    return fma(r, fma(e, e, e), r);
}
// 2^-k for the biased exponent field of a positive normal w = m 2^k: an exact rescaling factor
__device__ __forceinline__ double pow2_inv_of(double w)
{
    const int e = (__double2hiint(w) >> 20) & 0x7FF;
    return __hiloint2double((2046 - e) << 20, 0);
}


// EXACT: nx is a multiple of M (every chunk is full: no per-row bounds checks).  The coefficients {a_i, c_i}
// are staged in shared memory, chunk q at slots [q (M+1), q (M+1) + M]: one conflict-free LDS.128 per row.
__host__ __device__ constexpr int k3_coef_slots(int nx, int M) { return (nx / M + 2) * (M + 1); }

// Chunk boundaries.  With 64-byte tile rows (KW = 4) a quarter warp holds two chunks q, q+1 of the same four
// systems; their rows i0 + r are M rows = a multiple of 128 bytes apart, i.e. on the same 16 banks (ncu: 4.2-way
// conflicts on every tile access, 2000 of 5300 shared-memory wavefronts per tile).  SKEW = 1 starts the odd chunks
// one row later (even chunks have M+1 rows, odd ones M-1), so that at every unrolled step the two chunks touch
// rows of different parity = the two halves of the 32 banks.
constexpr int K3_SKEW = 0;   // measured: 6 % slower with 1 (one more step on the dependent chain costs more than the conflicts)
__host__ __device__ constexpr int k3_chunk_start(int q, int M, int skew, int nx, int pch)
{
    return q >= pch ? nx : ((q * M + skew * (q & 1) < nx - 1) ? q * M + skew * (q & 1) : nx - 1);
}

// rows per TMA box of the K3 tile gather (box = 8 ky x 1 kz x k3_box_rows(nx) planes), and the rows the
// boxes cover together (>= nx; the excess is out of bounds in i and arrives as zeros)
__host__ __device__ constexpr int k3_num_boxes(int nx) { return (nx + 255) / 256; }
// (an even number of rows: a box of 64-byte rows then starts on a 128-byte boundary of the shared-memory tile, as TMA requires)
__host__ __device__ constexpr int k3_box_rows(int nx) { return ((nx + k3_num_boxes(nx) - 1) / k3_num_boxes(nx) + 1) / 2 * 2; }
__host__ __device__ constexpr int k3_tile_rows(int nx) { return k3_num_boxes(nx) * k3_box_rows(nx); }

// KW = systems (consecutive ky) per CTA: 8 (128-byte rows), or 4 (64-byte rows; half the shared memory, so that
// two CTAs share an SM and one gathers while the other computes -- used when the 8-wide tile allows only one).
// TB = thread bound of the instantiation (KW times the largest number of chunks it is launched with).
template <int M, bool EXACT, int KW, int TB>
__global__ void __launch_bounds__(TB) k_solve_x(DevParams P, const __grid_constant__ CUtensorMap mapC, cplx* __restrict__ T)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar;
    const int nx = P.nx, PCH = blockDim.x / KW;
    // [k3_tile_rows(nx)][KW], 128-byte aligned by hand (TMA destination; the launch adds 128 bytes of slack)
    cplx* tile = reinterpret_cast<cplx*>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u)); // (offset form keeps the shared state space)
    double* red = reinterpret_cast<double*>(tile + (size_t)k3_tile_rows(nx) * KW); // 2 buffers x 5 arrays x [PCH][KW]
    double2* coef = reinterpret_cast<double2*>(red + 10 * PCH * KW);  // [nx + nx/M + 1] {a_i, c_i}, one pad slot per chunk
    const int nkt = P.ny / 8, ntile = P.ny / KW;
    const int kz = blockIdx.x / ntile, ky0 = (blockIdx.x % ntile) * KW;   // first ky of this CTA
    const int s = threadIdx.x % KW, q = threadIdx.x / KW;
    const int slot = q * KW + s, NS = PCH * KW;
    constexpr int SK = (KW == 4) ? K3_SKEW : 0;    // skewed chunk starts (k3_chunk_start)
    constexpr bool FULL = EXACT && SK == 0;        // every chunk has exactly M rows
    constexpr int NI = M - 1 + SK;                 // most interior rows of a chunk

    // gather the 8 columns C[kz][0..nx)[8 kyt .. 8 kyt + 8): TMA boxes of 128-byte rows, one mbarrier
    if (threadIdx.x == 0) {
        mbar_init(&bar, 1);
        fence_mbar_init();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const int nb = k3_num_boxes(nx), br = k3_box_rows(nx);
        const unsigned long long pol = l2_policy((P.hints & 1) ? 1 : 0);
        // the coefficient table (already in the shared-memory layout) rides on the same mbarrier as the tile
        const uint32_t coef_bytes = (uint32_t)(k3_coef_slots(nx, M) * sizeof(double2));
        mbar_expect_tx(&bar, (uint32_t)(nb * br * KW * sizeof(cplx)) + coef_bytes);
        for (int b = 0; b < nb; ++b) tma_load_3d_hint(tile + (size_t)b * br * KW, &mapC, ky0 * 2, b * br, kz, &bar, pol);
        bulk_load(coef, P.acp, coef_bytes, &bar);
        // the tile of the CTA that will take this one's place on the SM: HBM -> L2 now, so that its gather is an L2 hit
        const unsigned nxt = blockIdx.x + (unsigned)P.k3_prefetch;
        if (P.k3_prefetch > 0 && nxt < gridDim.x) {
            const int kz2 = nxt / ntile, ky2 = (nxt % ntile) * KW;
            for (int b = 0; b < nb; ++b) tma_prefetch_3d(&mapC, ky2 * 2, b * br, kz2);
        }
    }
    const double lam = __ldg(&P.lamy[ky0 + s]) + __ldg(&P.lamz[kz]);
    mbar_wait(&bar, 0);
    const bool cta_singular = (blockIdx.x == 0) && P.has_mean;
    const int i0 = k3_chunk_start(q, M, SK, nx, PCH);
    const int i1 = k3_chunk_start(q + 1, M, SK, nx, PCH) - 1; // interface row of this chunk
    const double2* mycoef = coef + q * (M + 1);
    auto ld_ac = [&](int i) -> double2 { return mycoef[i - i0]; };   // {a_i, c_i}, i0 <= i <= i1: one conflict-free LDS.128
    double* bA = red;
    double* bC = red + NS;
    double* bL = red + 2 * NS;
    double* bFr = red + 3 * NS;
    double* bFi = red + 4 * NS;
    double* nA = red + 5 * NS;
    double* nC = nA + NS;
    double* nL = nA + 2 * NS;
    double* nFr = nA + 3 * NS;
    double* nFi = nA + 4 * NS;

    constexpr int MI = (NI > 0) ? NI : 1;
    double G[MI], H[MI];
    double rA, rC, rL, rFr, rFi;
    {   // ONE elimination sweep over the chunk interior, in place (tile <- y), one reciprocal per row:
        //   x_i = y_i + g_i x_{i+1} + h_i E_{q-1},   g + h + t = 1.
        // Along the way the first interior row is expressed in the two interfaces by prefix products of g
        // (Pg = g_0 ... g_{r-1}):   x_{i0} = Y + Gq E_q + Hq E_{q-1},
        //   Y = sum Pg y_r,  Hq = sum Pg h_r,  Gq = g_0 ... g_last,  Tq = 1 - Gq - Hq = sum Pg t_r  (no cancellation)
        // -- what the interface above needs for its reduced row, without a second (upward) elimination.
        // The kernel is bound by the latency of this dependent chain (ncu: 16 warps per SM, short-scoreboard and
        // fixed-latency stalls), so the pivots are carried UNNORMALISED: with W = the product of the pivots so far,
        //   Hn = h W, Tn = t W, S = Hn + Tn, Yn = y W:
        //   W <- (c + lam) W + a S,  S <- a S + lam W,  Hn <- a Hn,  Tn <- a Tn + lam W,  Yn <- a Yn + f W
        // -- linear recurrences two operations deep, still sums of non-negatives (R9); the reciprocal of W and
        // everything normalised by it (g = c W'/W, h, t, y) is off the chain.  W grows by at most the largest pivot
        // per row; every 8 rows all carried quantities are rescaled by the exact power of two 2^-exponent(W).
        double Hn = 1.0, Tn = 0.0, S = 1.0, W = 1.0, Ynr = 0.0, Yni = 0.0;
        double h = 1.0, t = 0.0, yr = 0.0, yi = 0.0;
        double Pg = 1.0, Yr = 0.0, Yi = 0.0, Hq = 0.0, Tq = 0.0;
#pragma unroll
        for (int r = 0; r < NI; ++r) {
            const int i = i0 + r;
            if (FULL || i < i1) {
                if (r > 0 && r % 8 == 0) {
                    const double sc = pow2_inv_of(W);
                    W *= sc; S *= sc; Hn *= sc; Tn *= sc; Ynr *= sc; Yni *= sc;
                }
                const double2 ac = ld_ac(i);
                const double a = ac.x, c = ac.y;
                const cplx f = tile[i * KW + s];
                const double lw = lam * W;
                const double Wn = fma(c + lam, W, a * S);
                S = fma(a, S, lw);
                Hn = a * Hn;
                Tn = fma(a, Tn, lw);
                Ynr = fma(a, Ynr, f.x * W);
                Yni = fma(a, Yni, f.y * W);
                const double rw = fast_rcp(Wn);
                const double g = (c * W) * rw;
                W = Wn;
                h = Hn * rw;
                t = Tn * rw;
                yr = Ynr * rw;
                yi = Yni * rw;
                tile[i * KW + s] = mk(yr, yi);
                G[r] = g;
                H[r] = h;
                Yr = fma(Pg, yr, Yr);
                Yi = fma(Pg, yi, Yi);
                Hq = fma(Pg, h, Hq);
                Tq = fma(Pg, t, Tq);
                Pg *= g;
            }
        }
        if (q > 0) { // contribution to the interface row above (reduced row q-1); staged in the "next" buffer
            const double cb = mycoef[-(M + 1) + (i0 - 1 - k3_chunk_start(q - 1, M, SK, nx, PCH))].y;   // c of the interface row above
            nC[slot - KW] = cb * Pg;
            nL[slot - KW] = cb * Tq;
            nFr[slot - KW] = cb * Yr;
            nFi[slot - KW] = cb * Yi;
        }
        const double ab = ld_ac(i1).x;
        const cplx f = tile[i1 * KW + s];
        rA = ab * h;
        rL = fma(ab, t, lam);
        rFr = fma(ab, yr, f.x);
        rFi = fma(ab, yi, f.y);
    }
    __syncthreads();
    if (q < PCH - 1) {
        rC = nC[slot];
        rL += nL[slot];
        rFr += nFr[slot];
        rFi += nFi[slot];
    } else {
        rC = 0.0;
    }
    if (cta_singular && s == 0 && q == PCH - 1) { // pin the last unknown of the mean mode
        rA = 0.0; rC = 0.0; rL = 1.0; rFr = 0.0; rFi = 0.0;
    }
    // cancellation-free PCR over the PCH interface unknowns of each system.  Every row publishes itself
    // NORMALISED by its own diagonal (one reciprocal per row and level, before the exchange), so that the
    // elimination factors al = A / D(q-d), ga = C / D(q+d) need no reciprocal after the loads.
    for (int d = 1; d < PCH; d <<= 1) {
        const double rD = fast_rcp(rA + rC + rL);
        bA[slot] = rA * rD; bC[slot] = rC * rD; bL[slot] = rL * rD; bFr[slot] = rFr * rD; bFi[slot] = rFi * rD;
        __syncthreads();
        double A2 = 0.0, C2 = 0.0;
        if (q - d >= 0) {
            const int m = slot - KW * d;
            A2 = rA * bA[m];
            rL = fma(rA, bL[m], rL);
            rFr = fma(rA, bFr[m], rFr);
            rFi = fma(rA, bFi[m], rFi);
        }
        if (q + d < PCH) {
            const int m = slot + KW * d;
            C2 = rC * bC[m];
            rL = fma(rC, bL[m], rL);
            rFr = fma(rC, bFr[m], rFr);
            rFi = fma(rC, bFi[m], rFi);
        }
        rA = A2;
        rC = C2;
        // swap buffers
        double* tp;
        tp = bA; bA = nA; nA = tp;
        tp = bC; bC = nC; nC = tp;
        tp = bL; bL = nL; nL = tp;
        tp = bFr; bFr = nFr; nFr = tp;
        tp = bFi; bFi = nFi; nFi = tp;
    }
    {
        const double rr = fast_rcp(rA + rC + rL);
        const double er = rFr * rr, ei = rFi * rr;
        bFr[slot] = er;
        bFi[slot] = ei;
        __syncthreads();
        const double elr = (q > 0) ? bFr[slot - KW] : 0.0, eli = (q > 0) ? bFi[slot - KW] : 0.0;
        double xr = er, xi = ei;
        // T[kz][kyt][i][8]: the tile is contiguous in global memory.  All CTAs but the one holding the
        // mean mode store x straight from the back substitution (64/128-byte segments per row; the stores
        // drain while the next CTA of this SM already loads its tile).
        cplx* dst = T + ((size_t)kz * nkt + ky0 / 8) * (size_t)nx * 8 + (ky0 % 8);
        if (!cta_singular) {
            dst[i1 * 8 + s] = mk(xr, xi);
#pragma unroll
            for (int r = NI - 1; r >= 0; --r) {
                const int i = i0 + r;
                if (FULL || i < i1) {
                    const cplx y = tile[i * KW + s];
                    xr = fma(G[r], xr, fma(H[r], elr, y.x));
                    xi = fma(G[r], xi, fma(H[r], eli, y.y));
                    dst[i * 8 + s] = mk(xr, xi);
                }
            }
            return;
        }
        tile[i1 * KW + s] = mk(xr, xi);
#pragma unroll
        for (int r = NI - 1; r >= 0; --r) {
            const int i = i0 + r;
            if (FULL || i < i1) {
                const cplx y = tile[i * KW + s];
                xr = fma(G[r], xr, fma(H[r], elr, y.x));
                xi = fma(G[r], xi, fma(H[r], eli, y.y));
                tile[i * KW + s] = mk(xr, xi);
            }
        }
    }
    __syncthreads();
    if (cta_singular) { // zero dx-weighted mean for mode (0,0) = system s = 0 of this CTA
        if (s == 0) {
            double sr = 0.0, si = 0.0;
            for (int i = i0; i <= i1; ++i) {
                const double wgt = __ldg(&P.dxw[i]);
                const cplx x = tile[i * KW];
                sr = fma(x.x, wgt, sr);
                si = fma(x.y, wgt, si);
            }
            nFr[q] = sr;
            nFi[q] = si;
        }
        __syncthreads();
        if (s == 0) {
            double sr = 0.0, si = 0.0;
            for (int qq = 0; qq < PCH; ++qq) { sr += nFr[qq]; si += nFi[qq]; }
            sr *= P.inv_vol;
            si *= P.inv_vol;
            for (int i = i0; i <= i1; ++i) {
                cplx x = tile[i * KW];
                x.x -= sr;
                x.y -= si;
                tile[i * KW] = x;
            }
        }
        __syncthreads();
    }
    {   // the mean-mode CTA: contiguous store of the tile
        cplx* dst = T + ((size_t)kz * nkt + ky0 / 8) * (size_t)nx * 8 + (ky0 % 8);
        for (int e = threadIdx.x; e < nx * KW; e += blockDim.x) dst[(e / KW) * 8 + (e % KW)] = tile[e];
    }
}

// ------------------------------------------------------------------------------------------
// SURVEY.md 8(f1), fast path: the x-solve of a REAL field when every column has the SAME matrix (the implicit
// wall-normal step): all pivot quantities of k_solve_x's algorithm (two-sided chunk elimination, reduced
// interface system, PCR, back substitution) depend only on the row, so afid_xsolve_create evaluates them once
// on the host in long double and the kernel only runs the data recurrences:
//   up    yu <- (c rr)_i yu + (rr)_i f_i                 (UP[i]  = {c_i rr_i, rr_i},  rows i1-1 .. i0)
//   down  yd <- (a rr)_i yd + (rr)_i f_i ,  tile <- yd   (DN[i]  = {a_i rr_i, rr_i},  rows i0 .. i1-1)
//   F_q   = f_i1 + ab_q yd + cb_{q+1} yu_{q+1}           (CH[q]  = {ab_q, cb_q})
//   PCR   F_q <- F_q + al F_{q-d} + ga F_{q+d}           (PC[lev][q] = {al, ga}),  E_q = rrE_q F_q
//   back  x_i = y_i + G_i x_{i+1} + H_i E_{q-1}          (GH[i]  = {G_i, H_i})
// Tile = (line j, KW complex lanes = 2 KW real k columns) x all nx rows, rows a plane apart, gathered by TMA;
// thread (s, q) owns rows [qM, qM+M) of lane s, as in k_solve_x.  KW = 8 (128-byte rows) wherever the tile
// fits: 64-byte rows a plane apart run at 0.43 of the copy bandwidth, 128-byte rows at 0.5-0.63 (an L2
// prefetch of the full lines before the 64-byte gather made it slower).  The tables are read through L1.
// ------------------------------------------------------------------------------------------
struct XsTables {
    const double2* UP;   // [nx]
    const double2* DN;   // [nx]
    const double2* GH;   // [nx]
    const double2* CH;   // [PCH]  {ab_q, cb_q}
    const double* RE;    // [PCH]  1 / (A + C + L) of the fully reduced row
    const double2* PC;   // [nlev][PCH] {al, ga}
    int nlev;
};

template <int M, int KW>
__global__ void __launch_bounds__(64 * KW, (KW == 4) ? 3 : 1) k_xsolve_field(DevParams P, XsTables X, const __grid_constant__ CUtensorMap map, cplx* __restrict__ F)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar;
    const int nx = P.nx, PCH = blockDim.x / KW;
    cplx* tile = reinterpret_cast<cplx*>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));   // [k3_tile_rows(nx)][KW]
    cplx* red = tile + (size_t)k3_tile_rows(nx) * KW;                                                  // 2 x [PCH][KW]
    const int ntile = (P.nz / 2) / KW;
    const int j = blockIdx.x / ntile, c0 = (blockIdx.x % ntile) * KW;   // line j, first complex column
    const int s = threadIdx.x % KW, q = threadIdx.x / KW;
    const int slot = q * KW + s, NS = PCH * KW;
    if (threadIdx.x == 0) {
        mbar_init(&bar, 1);
        fence_mbar_init();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const int nb = k3_num_boxes(nx), br = k3_box_rows(nx);
        const unsigned long long pol = l2_policy((P.hints & 1) ? 1 : 0);
        mbar_expect_tx(&bar, (uint32_t)(nb * br * KW * sizeof(cplx)));
        for (int b = 0; b < nb; ++b) tma_load_3d_hint(tile + (size_t)b * br * KW, &map, c0 * 2, j, b * br, &bar, pol);
    }
    const int i0 = q * M;
    const int i1 = min(i0 + M, nx) - 1; // interface row of this chunk
    const double2 ch = __ldg(&X.CH[q]);
    mbar_wait(&bar, 0);
    cplx* my = tile + (size_t)i0 * KW + s;
    // upward: relation of the first interior row to the interface above (read only)
    double ur = 0.0, ui = 0.0;
#pragma unroll
    for (int r = M - 2; r >= 0; --r) {
        if (i0 + r < i1) {
            const double2 t = __ldg(&X.UP[i0 + r]);
            const cplx f = my[r * KW];
            ur = fma(t.x, ur, t.y * f.x);
            ui = fma(t.x, ui, t.y * f.y);
        }
    }
    if (q > 0) red[NS + slot - KW] = mk(ch.y * ur, ch.y * ui); // cb_q yu_q -> reduced row q-1 (staged in buffer 1)
    // downward, in place: tile <- y
    double dr = 0.0, di = 0.0;
#pragma unroll
    for (int r = 0; r < M - 1; ++r) {
        if (i0 + r < i1) {
            const double2 t = __ldg(&X.DN[i0 + r]);
            const cplx f = my[r * KW];
            dr = fma(t.x, dr, t.y * f.x);
            di = fma(t.x, di, t.y * f.y);
            my[r * KW] = mk(dr, di);
        }
    }
    double fr, fi;
    {
        const cplx f = tile[(size_t)i1 * KW + s];
        fr = fma(ch.x, dr, f.x);
        fi = fma(ch.x, di, f.y);
    }
    __syncthreads();
    if (q < PCH - 1) {
        const cplx t = red[NS + slot];
        fr += t.x;
        fi += t.y;
    }
    // PCR on the right-hand side only (the matrix part was done on the host)
    cplx* bA = red;
    cplx* bB = red + NS;
    for (int lev = 0, d = 1; lev < X.nlev; ++lev, d <<= 1) {
        __syncthreads();            // previous level's reads (and the staging reads above) are done
        bA[slot] = mk(fr, fi);
        __syncthreads();
        const double2 pc = __ldg(&X.PC[lev * PCH + q]);
        if (q - d >= 0) { const cplx m = bA[slot - KW * d]; fr = fma(pc.x, m.x, fr); fi = fma(pc.x, m.y, fi); }
        if (q + d < PCH) { const cplx m = bA[slot + KW * d]; fr = fma(pc.y, m.x, fr); fi = fma(pc.y, m.y, fi); }
        cplx* tp = bA; bA = bB; bB = tp;
    }
    const double re = __ldg(&X.RE[q]);
    double xr = fr * re, xi = fi * re;
    __syncthreads();
    bA[slot] = mk(xr, xi);
    __syncthreads();
    const cplx el = (q > 0) ? bA[slot - KW] : mk(0.0, 0.0);
    // back substitution with direct stores: row i of the tile = F[i][j][2 c0 .. 2 c0 + 2 KW)
    cplx* dst = F + (size_t)j * (P.nz / 2) + c0 + s;
    const size_t rstride = (size_t)P.ny * (P.nz / 2);
    dst[(size_t)i1 * rstride] = mk(xr, xi);
#pragma unroll
    for (int r = M - 2; r >= 0; --r) {
        if (i0 + r < i1) {
            const double2 gh = __ldg(&X.GH[i0 + r]);
            const cplx y = my[r * KW];
            xr = fma(gh.x, xr, fma(gh.y, el.x, y.x));
            xi = fma(gh.x, xi, fma(gh.y, el.y, y.y));
            dst[(size_t)(i0 + r) * rstride] = mk(xr, xi);
        }
    }
}

// ------------------------------------------------------------------------------------------
// maximum CFL number, the paper's Listing 1 "CalcMaxCFL":
//   cflm = max(1e-8, max over cells 0.5 (|w(k)+w(k+1)|/dz + |v(j)+v(j+1)|/dy + |u(i)+u(i+1)|/dx_i))
// (AFiD's dz, dy, udx3m are inverse spacings).  Same CTA map as K6: (i, 4 lines), four 16-byte pairs per
// thread per batch; plane i+1 of u and line j+1 of v are L2 hits.  Non-negative doubles order like
// their bit patterns, so the grid-wide maximum is one atomicMax on the 64-bit pattern per CTA.  The whole
// reduction runs on the bit patterns: a NaN (from a blown-up field) has the largest pattern and therefore
// reaches the result instead of being dropped by fmax (a time stepper must see it).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long cfl_bits(double q)   // q >= 0 or NaN
{
    return (unsigned long long)__double_as_longlong(q) & 0x7FFFFFFFFFFFFFFFull;
}
__device__ __forceinline__ unsigned long long umax64(unsigned long long a, unsigned long long b) { return a > b ? a : b; }
__global__ void k_cfl_init(double* __restrict__ cfl) { *cfl = 0.00000001; }

__device__ __forceinline__ double2 ldcg2(const double* p)   // L2 only: data another SM wrote during this launch
{
    double2 r;
    asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ double ldcg1(const double* p)
{
    double r;
    asm volatile("ld.global.cg.f64 %0, [%1];" : "=d"(r) : "l"(p));
    return r;
}

// Listing 1 over the cells of ONE line (i, j, all k) per thread row: thread x takes the cell pairs kp = x, x + TX, ...
// in batches of U.  Returns the bit pattern of the thread's maximum.  CG: the loads bypass L1 (the fused kernel reads
// what other SMs wrote a moment ago; L1 may still hold the uncorrected lines).
template <bool CG, int U>
__device__ __forceinline__ unsigned long long cfl_line(const DevParams& P, const double* __restrict__ u, const double* __restrict__ v,
                                                       const double* __restrict__ w, int i, int j)
{
    constexpr int TX = K6_TX;
    const int jp = (j + 1 == P.ny) ? 0 : j + 1;
    const size_t plane = (size_t)P.ny * P.nz;
    const size_t ol = ((size_t)i * P.ny + j) * P.nz;
    const double *ul = u + ol, *vl = v + ol, *wl = w + ol;
    const double* vp = v + ((size_t)i * P.ny + jp) * P.nz;
    const int nzh2 = P.nz / 2;
    const double rdx = __ldg(&P.rdx[i]), rdy = P.rdy, rdz = P.rdz;
    auto ld2 = [](const double* q) -> double2 { return CG ? ldcg2(q) : ldg2(q); };
    auto ld1 = [](const double* q) -> double { return CG ? ldcg1(q) : __ldg(q); };
    unsigned long long best = 0ull;
    for (int k0 = threadIdx.x; k0 < nzh2; k0 += TX * U) {
        double2 u0[U], u1[U], v0[U], v1[U], w0[U];
        double wn[U];
#pragma unroll
        for (int r = 0; r < U; ++r) {
            const int kp = k0 + r * TX;
            if (kp < nzh2) {
                u0[r] = ld2(ul + 2 * kp);
                u1[r] = ld2(ul + plane + 2 * kp);
                v0[r] = ld2(vl + 2 * kp);
                v1[r] = ld2(vp + 2 * kp);
                w0[r] = ld2(wl + 2 * kp);
                wn[r] = ld1(wl + (kp == nzh2 - 1 ? 0 : 2 * kp + 2));
            }
        }
#pragma unroll
        for (int r = 0; r < U; ++r) {
            const int kp = k0 + r * TX;
            if (kp < nzh2) {
                const double qa = fabs((w0[r].x + w0[r].y) * rdz) + fabs((v0[r].x + v1[r].x) * rdy) + fabs((u0[r].x + u1[r].x) * rdx);
                const double qb = fabs((w0[r].y + wn[r]) * rdz) + fabs((v0[r].y + v1[r].y) * rdy) + fabs((u0[r].y + u1[r].y) * rdx);
                best = umax64(best, umax64(cfl_bits(qa * 0.5), cfl_bits(qb * 0.5)));
            }
        }
    }
    return best;
}
// maximum over the CTA, one atomicMax on the bit pattern (s_max: one slot per warp; the caller synchronises before reuse)
__device__ __forceinline__ void cfl_block_max(unsigned long long best, unsigned long long* s_max, double* __restrict__ cfl)
{
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) best = umax64(best, __shfl_xor_sync(0xffffffffu, best, d));
    const int tid = threadIdx.y * K6_TX + threadIdx.x;
    if ((tid & 31) == 0) s_max[tid >> 5] = best;
    __syncthreads();
    if (tid == 0) {
        for (int k = 1; k < K6_JL * K6_TX / 32; ++k) best = umax64(best, s_max[k]);
        atomicMax(reinterpret_cast<unsigned long long*>(cfl), best);
    }
}

__global__ void __launch_bounds__(K6_JL* K6_TX) k_max_cfl(DevParams P, const double* __restrict__ u, const double* __restrict__ v,
                                                          const double* __restrict__ w, double* __restrict__ cfl)
{
    __shared__ unsigned long long s_max[K6_JL * K6_TX / 32];
    int i, jg;
    k6_item_to_ij((int)blockIdx.x, P.nx, P.ny / K6_JL, i, jg);
    cfl_block_max(cfl_line<false, K6_U>(P, u, v, w, i, jg * K6_JL + threadIdx.y), s_max, cfl);
}

// ------------------------------------------------------------------------------------------
// SURVEY.md 8(f3), fused form: the correction (K6) with Listing 1's maximum taken over the CORRECTED field in
// the same launch -- no second pass over u, v, w through HBM.  A cell's value needs the corrected u(i+1), v(j+1),
// w(k+1), which belong to other CTAs' lines and are overwritten in place, so the reduction cannot ride in the
// correcting CTA's registers.  Instead one persistent launch hands out tickets: ticket t corrects item t (the
// CTA order of k_correct) and then reduces the cells of item t - lag, whose lines were corrected `lag` tickets
// ago and are still in L2 (lag = resident CTAs + 16 items: < 50 MB of u, v, w at C4).  The reduce step owns the
// lines JL jg - 1 .. JL jg + JL - 2 (one line down, so that v(j+1) stays inside the chunk that was just
// corrected; the last group also takes line ny - 1, whose neighbour is line 0) and waits for the "done" flags
// of the (at most five) items that wrote what it reads.  Every wait is for an EARLIER ticket, whose correction
// part never waits: no deadlock whatever order the CTAs are scheduled in.  sync[0] = ticket counter,
// sync[1 + s] = item s corrected (both zeroed by the host before the launch).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int ld_acquire_i32(const int* p)
{
    int r;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(r) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st_release_i32(int* p, int v) { asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory"); }

// U, MINB: cell pairs per load batch and CTAs per SM the register allocation is capped for.  <4, 1> (236 registers, one
// CTA per SM) is the measured default; <2, 2> lets one CTA's reduce step overlap the other's correction (hint bit 32).
template <int U, int MINB>
__global__ void __launch_bounds__(K6_JL* K6_TX, MINB) k_correct_cfl(DevParams P, const double* __restrict__ p, double* __restrict__ u, double* __restrict__ v,
                                                              double* __restrict__ w, double* __restrict__ pacc, double* __restrict__ cfl, int* __restrict__ sync,
                                                              int lag)
{
    constexpr int JL = K6_JL, TX = K6_TX;
    __shared__ unsigned long long s_max[JL * TX / 32];
    __shared__ int s_tk;
    const int tid = threadIdx.y * TX + threadIdx.x;
    const int ngrp = P.ny / JL, nitems = P.nx * ngrp;
    int* done = sync + 1;
    // the uncorrected u, v, w are read once: evict first; hint bit 2: the corrected lines evict last (kept for the reduce step)
    const unsigned long long pol_in = l2_policy((P.hints & 4) ? 0 : 1), pol_out = l2_policy((P.hints & 2) ? 2 : 0);
    int nxt = 0;
    if (tid == 0) nxt = atomicAdd(&sync[0], 1);
#pragma unroll 1
    for (;;) {
        if (tid == 0) {
            s_tk = nxt;
            nxt = atomicAdd(&sync[0], 1);   // the next ticket is fetched one item ahead: its latency hides behind this item
        }
        __syncthreads();
        const int tk = s_tk;
        if (tk >= nitems + lag) break;
        if (tk < nitems) {
            int i, jg;
            k6_item_to_ij(tk, P.nx, ngrp, i, jg);
            k6_correct_item<U>(P, p, u, v, w, i, jg, pacc, nullptr, pol_in, pol_out);
            __syncthreads();
            if (tid == 0) {
                __threadfence();
                st_release_i32(&done[tk], 1);
            }
        }
        const int sc = tk - lag;
        unsigned long long best = 0ull;
        if (sc >= 0) {
            int i, jg;
            k6_item_to_ij(sc, P.nx, ngrp, i, jg);
            if (tid < 5) {   // the items that wrote what this step reads
                const int di = (tid & 1) ? i + 1 : i;
                const int dg = (tid == 4) ? 0 : ((tid & 2) ? jg - 1 : jg);
                const bool need = (di < P.nx) && (dg >= 0) && (tid < 4 || (jg == ngrp - 1 && di == i));
                if (need) {
                    const int* f = &done[k6_ij_to_item(di, dg, P.nx, ngrp)];
                    while (ld_acquire_i32(f) == 0) __nanosleep(64);
                }
            }
            __syncthreads();
            const int npass = (jg == ngrp - 1) ? 2 : 1;   // (the last group also takes line ny - 1)
#pragma unroll 1
            for (int pass = 0; pass < npass; ++pass) {
                const int j = (pass == 0) ? jg * JL - 1 + (int)threadIdx.y : ((threadIdx.y == 0) ? P.ny - 1 : -1);
                if (j >= 0) best = umax64(best, cfl_line<true, U>(P, u, v, w, i, j));
            }
        }
        cfl_block_max(best, s_max, cfl);
        __syncthreads();   // s_tk and s_max are rewritten by the next step
    }
}

} // namespace afid
