// panel.cuh -- SURVEY.md 8a row a1: unblocked Householder factorisation of an IB-wide inner
// panel, the latency-bound heart of a blocked dgeqrf (Eq. 2).
//
// Design (differs from a LAPACK geqr2 loop, same arithmetic): the m_k x IB inner panel is
// spread over G co-resident CTAs (cooperative launch); every thread keeps RPT rows x IB
// columns in REGISTERS for the whole kernel.  Column j needs sigma^2 = sum x_i^2 and
// w_c = v^T a_c; both follow from s_c = sum_{i>j} x_i a_c[i] (c = 0..IB-1, one pass, before
// beta is known):  sigma^2 = s_j,  w_c = a_c[j] + s_c/(alpha-beta).  The same pass also yields
// V[:,0:j]^T v_j, so the inner T factor comes for free.  Hence ONE grid-wide reduction per
// column: warp-shuffle transpose-reduce -> shared memory -> per-CTA partial published in global
// memory with the "LL" flag-in-data protocol (every 8-byte store carries 4 bytes of payload and
// the 4-byte step number, so a reader that sees the right step number in both halves has the
// value: data exchange and grid barrier are ONE L2 round trip, no fence, no counter) -> every
// CTA sums the G partials in the same fixed order (bit-identical scalars everywhere,
// deterministic run to run).
// The update by reflector j and the dot products for column j+1 are fused into one register pass.
#pragma once
#include "common.cuh"
#include "kernels.h"

namespace ctqr {

// Sum IB per-thread values across the 32 lanes of a warp.  On return lane l holds in v[0] the
// warp total of column (l * IB) / 32 (IB = 32: column l; IB = 16: l>>1; IB = 8: l>>2).
template <typename T, int IB>
__device__ __forceinline__ void warp_transpose_reduce(T (&v)[IB], int lane) {
    int k = IB / 2;
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        if (k >= 1) {
            const bool upper = (lane & off) != 0;
#pragma unroll
            for (int i = 0; i < IB / 2; ++i) {
                if (i < k) {
                    T send = upper ? v[i] : v[i + k];
                    T keep = upper ? v[i + k] : v[i];
                    v[i] = keep + shfl_xor(send, off);
                }
            }
            k >>= 1;
        } else {
            v[0] = v[0] + shfl_xor(v[0], off);
        }
    }
}

// ---- LL slots: one 16-byte slot per value: {lo, seq, hi, seq} (fp32 uses lo only) -------------
__device__ __forceinline__ void ll_store(uint4* slot, double v, unsigned seq) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    asm volatile("st.volatile.global.v4.u32 [%0], {%1, %2, %3, %2};\n" ::"l"(slot), "r"((unsigned)b), "r"(seq),
                 "r"((unsigned)(b >> 32)) : "memory");
}
__device__ __forceinline__ void ll_store(uint4* slot, float v, unsigned seq) {
    asm volatile("st.volatile.global.v4.u32 [%0], {%1, %2, %1, %2};\n" ::"l"(slot), "r"(__float_as_uint(v)), "r"(seq) : "memory");
}
__device__ __forceinline__ uint4 ll_load(const uint4* slot) {
    uint4 r;
    asm volatile("ld.volatile.global.v4.u32 {%0, %1, %2, %3}, [%4];\n" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(slot) : "memory");
    return r;
}
template <typename T> __device__ __forceinline__ T ll_value(uint4 r);
template <> __device__ __forceinline__ double ll_value<double>(uint4 r) {
    return __longlong_as_double((long long)(((unsigned long long)r.z << 32) | r.x));
}
template <> __device__ __forceinline__ float ll_value<float>(uint4 r) { return __uint_as_float(r.x); }
// spin until the slot carries step `seq`, return its value
template <typename T>
__device__ __forceinline__ T ll_wait(const uint4* slot, unsigned seq) {
    uint4 r = ll_load(slot);
    while (r.y != seq || r.w != seq) r = ll_load(slot);
    return ll_value<T>(r);
}

template <typename T, int IB, int RPT, int NT>
__global__ void __launch_bounds__(NT, 1) panel_geqr2_kernel(PanelArgs<T> p) {
    static_assert(IB == 8 || IB == 16 || IB == 32, "IB");
    constexpr int NW = NT / 32;
    constexpr int NG = NT / IB;                 // reducer groups for the cross-CTA sum
    constexpr int LPC = 32 / IB;                // lanes per column after the warp reduce
    __shared__ T sh_warp[NW][IB];
    __shared__ T sh_red[NG][IB];
    __shared__ T sh_tw[IB];                     // c > j: tau*w_c
    __shared__ T sh_scal[4];                    // denom, beta, tau, flag(sigma2 != 0)
    __shared__ T sh_T[IB][IB + 1];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cta = blockIdx.x, G = gridDim.x;
    const int ibw = p.ibw;
    T* __restrict__ A = p.A;

    int64_t row[RPT];
    T a[RPT][IB];
#pragma unroll
    for (int q = 0; q < RPT; ++q) {
        row[q] = p.jb + ((int64_t)q * G + cta) * NT + tid;
#pragma unroll
        for (int c = 0; c < IB; ++c)
            a[q][c] = (row[q] < p.m && c < ibw) ? A[row[q] + (p.jb + c) * p.lda] : T(0);
    }
    if (cta == 0)
        for (int i = tid; i < IB * (IB + 1); i += NT) (&sh_T[0][0])[i] = T(0);

    // slots: [parity][G + 1][IB]; record G of a parity is the pivot row published by CTA 0
    uint4* slots = reinterpret_cast<uint4*>(p.part);

    // Reduce acc[] over the whole grid; afterwards warp 0 lane c (< IB) holds s_c and rj_c.
    // `pivot` (CTA 0 only): thread tid < IB passes its pivot-row entry to publish.
    auto grid_reduce = [&](T (&acc)[IB], int step, T pivot_val, bool has_pivot, T& s_out, T& rj_out) {
        const int par = step & 1;
        const unsigned seq = p.bar_base + (unsigned)step + 1u;
        uint4* base = slots + (size_t)par * (G + 1) * IB;
        if (has_pivot) ll_store(base + (size_t)G * IB + (tid % IB), pivot_val, seq);
        warp_transpose_reduce<T, IB>(acc, lane);
        if ((lane % LPC) == 0) sh_warp[warp][lane / LPC] = acc[0];
        __syncthreads();
        if (tid < IB) {
            T t = sh_warp[0][tid];
#pragma unroll
            for (int w = 1; w < NW; ++w) t += sh_warp[w][tid];
            ll_store(base + (size_t)cta * IB + tid, t, seq);
        }
        {
            // fixed summation order (same in every CTA); each thread waits for its own slots
            // the loads of a batch are issued before the first flag is examined; a slot that is
            // not there yet is re-polled individually
            const int c = tid % IB, grp = tid / IB;
            constexpr int MAXB = 4;
            T t = T(0);
            for (int b0 = grp; b0 < G; b0 += NG * MAXB) {
                uint4 r[MAXB];
#pragma unroll
                for (int i = 0; i < MAXB; ++i) {
                    const int b = b0 + i * NG;
                    if (b < G) r[i] = ll_load(base + (size_t)b * IB + c);
                }
#pragma unroll
                for (int i = 0; i < MAXB; ++i) {
                    const int b = b0 + i * NG;
                    if (b < G) {
                        while (r[i].y != seq || r[i].w != seq) r[i] = ll_load(base + (size_t)b * IB + c);
                        t += ll_value<T>(r[i]);
                    }
                }
            }
            sh_red[grp][c] = t;
        }
        __syncthreads();
        if (tid < IB) {
            T t = sh_red[0][tid];
#pragma unroll
            for (int gI = 1; gI < NG; ++gI) t += sh_red[gI][tid];
            s_out = t;
            rj_out = ll_wait<T>(base + (size_t)G * IB + tid, seq);
        }
    };

    // The column loop is NOT unrolled (a fully unrolled IB = 32 body is ~350 KB of SASS and the
    // kernel was instruction-fetch bound: ncu "no_instruction" stall 11.6 of 17 cycles per issue).
    // To keep every register index a compile-time constant anyway, the register tile is ROTATED by
    // one column per iteration: at the top of iteration j, position c of a[q][.] holds panel column
    // (j + c) mod IB, i.e. position 0 is always the current column, positions 1 .. ibw-1-j the
    // columns still to be updated, and the finished reflectors sit at the high positions (they are
    // still needed: the same dot-product pass yields V[:,0:j]^T v_j for the inner T factor).
    T s_c = T(0), rj_c = T(0);
    {
        // dots for column 0: acc[c] = sum over own rows strictly below the pivot row jb
        T acc[IB];
#pragma unroll
        for (int c = 0; c < IB; ++c) acc[c] = T(0);
#pragma unroll
        for (int q = 0; q < RPT; ++q) {
            const bool below = row[q] > p.jb;
            const T x = below ? a[q][0] : T(0);
#pragma unroll
            for (int c = 0; c < IB; ++c) acc[c] = fma(x, a[q][c], acc[c]);
        }
        // pivot row of column 0 = row jb, held by CTA 0 / thread 0 / q = 0
        if (cta == 0 && tid == 0) {
            const unsigned seq0 = p.bar_base + 1u;
#pragma unroll
            for (int c = 0; c < IB; ++c) ll_store(slots + (size_t)G * IB + c, a[0][c], seq0);
        }
        grid_reduce(acc, 0, T(0), false, s_c, rj_c);
    }

#pragma unroll 1
    for (int j = 0; j < ibw; ++j) {
        const int nact = ibw - 1 - j;          // positions 1 .. nact are columns still to be updated
        // ---- (2) scalars of reflector j (warp 0, lane = position; identical in every CTA) ----
        if (warp == 0) {
            const T alpha = __shfl_sync(0xffffffffu, rj_c, 0);
            const T sigma2 = __shfl_sync(0xffffffffu, s_c, 0);
            T beta = alpha, tauj = T(0), denom = T(1);
            const bool nz = sigma2 != T(0);
            if (nz) {
                T nrm = Num<T>::sqrt(fma(alpha, alpha, sigma2));
                beta = (alpha >= T(0)) ? -nrm : nrm;
                tauj = Num<T>::div(beta - alpha, beta);
                denom = alpha - beta;
            }
            // g = pivot-row entry + s/denom: active positions give w_c, finished ones (V^T v_j)_c
            const T gc = nz ? rj_c + Num<T>::div(s_c, denom) : T(0);
            if (lane < IB) sh_tw[lane] = (lane >= 1 && lane <= nact) ? tauj * gc : T(0);
            if (lane == 0) { sh_scal[0] = denom; sh_scal[1] = beta; sh_scal[2] = tauj; sh_scal[3] = nz ? T(1) : T(0); }
            if (cta == 0) {
                // inner T: T[0:j, j] = -tau_j * T[0:j,0:j] * g[0:j],  T[j][j] = tau_j
                // (panel column b < j sits at position b - j + IB)
                T sum = T(0);
                for (int b = 0; b < j; ++b) {
                    const T gb = __shfl_sync(0xffffffffu, gc, (b - j + IB) & 31);
                    if (lane < j && b >= lane) sum = fma(sh_T[lane][b], gb, sum);
                }
                __syncwarp();
                if (lane < j) sh_T[lane][j] = -tauj * sum;
                if (lane == j) sh_T[j][j] = tauj;
                if (lane == 0) p.tau[p.jb + j] = tauj;
            }
        }
        __syncthreads();
        const T denom = sh_scal[0], beta = sh_scal[1];
        const bool nz = sh_scal[3] != T(0);
        const volatile T* tw = sh_tw;      // re-read per use: keeps IB values out of the register file
        // ---- (3) apply reflector j to own rows, rotate, dots for column j+1 ----
        T acc[IB];
#pragma unroll
        for (int c = 0; c < IB; ++c) acc[c] = T(0);
        const int64_t piv = p.jb + j;
#pragma unroll
        for (int q = 0; q < RPT; ++q) {
            if (nz) {
                if (row[q] > piv) {
                    const T v = Num<T>::div(a[q][0], denom);
                    a[q][0] = v;
#pragma unroll
                    for (int c = 1; c < IB; ++c) a[q][c] = fma(-tw[c], v, a[q][c]);
                } else if (row[q] == piv) {
                    a[q][0] = beta;
#pragma unroll
                    for (int c = 1; c < IB; ++c) a[q][c] -= tw[c];
                }
            }
            {
                const T t0 = a[q][0];
#pragma unroll
                for (int c = 0; c + 1 < IB; ++c) a[q][c] = a[q][c + 1];
                a[q][IB - 1] = t0;
            }
            const bool below = row[q] > piv + 1;
            const T x = below ? a[q][0] : T(0);
#pragma unroll
            for (int c = 0; c < IB; ++c) acc[c] = fma(x, a[q][c], acc[c]);
        }
        if (j + 1 < ibw) {
            // pivot row of column j+1 = row jb+j+1, held by CTA 0 / thread j+1 / q = 0
            if (cta == 0 && tid == j + 1) {
                const unsigned seqn = p.bar_base + (unsigned)(j + 1) + 1u;
                uint4* rb = slots + ((size_t)((j + 1) & 1) * (G + 1) + G) * IB;
#pragma unroll
                for (int c = 0; c < IB; ++c) ll_store(rb + c, a[0][c], seqn);
            }
            grid_reduce(acc, j + 1, T(0), false, s_c, rj_c);
        }
    }
    // undo the rotation (ibw rotations done; IB - ibw more bring every column back to its index)
#pragma unroll 1
    for (int r = ibw; r < IB; ++r) {
#pragma unroll
        for (int q = 0; q < RPT; ++q) {
            const T t0 = a[q][0];
#pragma unroll
            for (int c = 0; c + 1 < IB; ++c) a[q][c] = a[q][c + 1];
            a[q][IB - 1] = t0;
        }
    }

    // ---- write back: V below the diagonal, explicit 0/1 on and above it; R to Rd ----
    const int64_t off = p.jb - p.j0;    // position of this inner block inside the panel
#pragma unroll
    for (int q = 0; q < RPT; ++q) {
        if (row[q] >= p.m) continue;
        const bool diagblk = (cta == 0 && q == 0 && tid < IB);
#pragma unroll
        for (int c = 0; c < IB; ++c) {
            if (c >= ibw) continue;
            T val = a[q][c];
            if (diagblk && c >= tid) {
                p.Rd[(off + tid) + (off + c) * (int64_t)p.ldrd] = val;
                val = (c == tid) ? T(1) : T(0);
            }
            A[row[q] + (p.jb + c) * p.lda] = val;
        }
    }
    // rows j0 .. jb-1 of these columns are finished R entries of the panel's diagonal block
    if (cta == G - 1) {
        const int nr = (int)off;
        for (int i = tid; i < nr * ibw; i += NT) {
            int r = i % nr, c = i / nr;
            T* src = &A[(p.j0 + r) + (p.jb + c) * p.lda];
            p.Rd[r + (off + c) * (int64_t)p.ldrd] = *src;
            *src = T(0);
        }
    }
    if (cta == 0) {
        __syncthreads();
        for (int i = tid; i < IB * IB; i += NT) {
            const int r = i % IB, c = i / IB;
            if (r < ibw && c < ibw) p.Tin[r + (size_t)c * p.ldtin] = sh_T[r][c];
        }
    }
}

}  // namespace ctqr
