// fd6_kernels_tiled.cuh — FD_VARIANT_TILED / FD_VARIANT_PAIRED: the fast derivative/update kernel
// (DESIGN.md "Kernels").  One template, three value types: float, double, and V2 (two fp32 cells per value,
// packed FFMA2/FADD2/FMUL2 arithmetic — the paired layout).
//
// One CTA owns a TX x TY column of values and marches along z through a chunk of planes.
//   in   plane t of the four fields + radius-3 halo: ONE 4-D TMA box copy (cp.async.bulk.tensor, mbarrier
//        complete_tx) into an NS-deep ring of stages; the w values of the output plane: one more box copy into
//        a 4-deep ring (only on substeps that read w), so no thread waits on a global load.  A stage is handed
//        back to the producer thread through an "empty" mbarrier on which every warp arrives once it is done
//        with the plane, so there is no CTA-wide barrier in the loop.
//   out  F_out, w (and div u) go straight from registers to global memory: a warp writes one 256-byte row
//        segment per array.  (Staging them in shared memory for TMA box stores was measured 5-11 % slower: the
//        kernel is bound by shared-memory bandwidth.)
// Each thread owns one column and keeps everything that couples planes thread-private:
//   win[f][8]   sliding window of its own column along z                     -> D1z, D2z          (Eq. 6, 7)
//               (8-byte value types: in TENSOR MEMORY, one tcgen05.st of the new plane and one 16-column
//               tcgen05.ld per field and plane; plain fp32: in registers)
//   lin[i][8]   accumulator ring of everything of dt*rhs_i that is known when a plane is staged: the in-plane
//               second derivatives (D2x, D2y, Dxy), the in-plane part of the nonlinear terms, and the mixed
//               derivatives that involve z (Eq. 8), which are formed from the in-plane differences
//               f(x+m) - f(x-m) that D1x / D1y need anyway:  Dxz f(z) = sum_m c_m [dx_m f(z+m) - dx_m f(z-m)],
//               so plane t scatters +-c_m dx_m into the ring slots of outputs t-m and t+m (no extra loads)
//   and parks in TENSOR MEMORY (tcgen05.st / tcgen05.ld; idle otherwise, there is no tensor-core work here) the
//   six in-plane quantities that multiply z derivatives, until their plane is the centre three planes later.
// Output plane z = t-3 is finished (Eq. 1-3) and updated (Eq. 10) when plane t = z+3 has been consumed.
// dt is folded into the velocity-derivative coefficients, so the kernel forms dt*rhs directly.
// The accumulation order of every output depends only on relative plane index, never on the position in a
// tile or chunk, so periodic-shift equivariance stays bitwise.
// PATH55 = false is pass 1 of the 19-point path (no mixed derivatives, dt*div u written, Eq. 14-16).
#pragma once
#include <cuda.h>

#include "fd6_tiled_host.cuh"

namespace fd6 {

// ---- mbarrier / TMA primitives (PTX ISA: mbarrier, cp.async.bulk.tensor) --------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// All helpers take 32-bit shared-window addresses, formed once per kernel from the base of the dynamic
// shared memory, so that the plane loop holds no generic-to-shared conversions.
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1, int c2, int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(dst),
        "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}

// ---- tensor memory as a per-thread delay line (tcgen05.st / tcgen05.ld, shape 32x32b: lane = thread of the
// warp's quadrant, consecutive 32-bit columns).  TMEM is otherwise idle in this kernel (no tensor-core work);
// parking the six delayed in-plane values of the last three planes there frees 36 registers per thread.
template <int N>
__device__ __forceinline__ void tmem_st(uint32_t taddr, const uint32_t* r) {
    static_assert(N == 2 || N == 4 || N == 8, "chunk size");
    if constexpr (N == 8)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]),
                     "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
                     : "memory");
    else if constexpr (N == 4)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3])
                     : "memory");
    else
        asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(r[0]), "r"(r[1]) : "memory");
}
template <int N>
__device__ __forceinline__ void tmem_ld(uint32_t taddr, uint32_t* r) {
    static_assert(N == 2 || N == 4 || N == 8, "chunk size");
    if constexpr (N == 8)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                     : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                     : "r"(taddr)
                     : "memory");
    else if constexpr (N == 4)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr) : "memory");
    else
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t* r) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
}
// Results of tcgen05.ld may be used only after tcgen05.wait::ld.  The *_nc variants carry no "memory" clobber (so the
// compiler may move shared-memory loads across them; volatile asm statements keep their order among themselves);
// instead the loaded registers are passed through tmem_fence*, an empty volatile asm placed after the wait, so that
// every consumer depends on it.
__device__ __forceinline__ void tmem_ld16_nc(uint32_t taddr, uint32_t* r) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld8_nc(uint32_t taddr, uint32_t* r) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld4_nc(uint32_t taddr, uint32_t* r) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr));
}
__device__ __forceinline__ void tmem_st2_nc(uint32_t taddr, const uint32_t* r) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(r[0]), "r"(r[1]));
}
__device__ __forceinline__ void tmem_st8_nc(uint32_t taddr, const uint32_t* r) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]),
                 "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]));
}
__device__ __forceinline__ void tmem_st4_nc(uint32_t taddr, const uint32_t* r) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]));
}
__device__ __forceinline__ void tmem_wait_ld_nc() { asm volatile("tcgen05.wait::ld.sync.aligned;"); }
__device__ __forceinline__ void tmem_wait_st_nc() { asm volatile("tcgen05.wait::st.sync.aligned;"); }
__device__ __forceinline__ void tmem_fence16(uint32_t* r) {
    asm volatile("" : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]), "+r"(r[8]), "+r"(r[9]),
                      "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15]));
}
__device__ __forceinline__ void tmem_fence4(uint32_t* r) { asm volatile("" : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3])); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// six values of T <-> 6 * sizeof(T) / 4 registers
template <class T>
struct Regs6 {
    static constexpr int N = 6 * (int)sizeof(T) / 4;
    static __device__ __forceinline__ void pack(const T v[6], uint32_t* r) {
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            if constexpr (sizeof(T) == 4) {
                r[i] = __float_as_uint(*reinterpret_cast<const float*>(&v[i]));
            } else {
                const uint2 u = *reinterpret_cast<const uint2*>(&v[i]);
                r[2 * i] = u.x;
                r[2 * i + 1] = u.y;
            }
        }
    }
    static __device__ __forceinline__ void unpack(const uint32_t* r, T v[6]) {
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            if constexpr (sizeof(T) == 4) {
                const float f = __uint_as_float(r[i]);
                v[i] = *reinterpret_cast<const T*>(&f);
            } else {
                const uint2 u = make_uint2(r[2 * i], r[2 * i + 1]);
                v[i] = *reinterpret_cast<const T*>(&u);
            }
        }
    }
    static __device__ __forceinline__ void store(uint32_t taddr, const T v[6]) {
        uint32_t r[N];
        pack(v, r);
        if constexpr (N == 12) {
            tmem_st<8>(taddr, r);
            tmem_st<4>(taddr + 8, r + 8);
        } else {
            tmem_st<4>(taddr, r);
            tmem_st<2>(taddr + 4, r + 4);
        }
    }
    static __device__ __forceinline__ void load(uint32_t taddr, T v[6]) {
        uint32_t r[N];
        if constexpr (N == 12) {
            tmem_ld<8>(taddr, r);
            tmem_ld<4>(taddr + 8, r + 8);
        } else {
            tmem_ld<4>(taddr, r);
            tmem_ld<2>(taddr + 4, r + 4);
        }
        tmem_wait_ld();
        unpack(r, v);
    }
};

// TX x TY threads; a thread owns RY vertically adjacent columns (rows cj .. cj+RY-1), so the tile is TX x (TY*RY).
// FORCE: the forcing term of Eq. 2 is added (a separate instantiation, so the unforced kernel pays nothing).
// MODE: what the RK update of the launch touches, known at compile time so that the plane loop holds no runtime
// predicates on it: bit 0 = w is read (alpha != 0), bit 1 = w is written, bit 2 = F_out is written.  The four modes
// in use: 6 = substep 1 (alpha_1 = 0: w not read), 7 = substep 2, 5 = substep 3 (its w is never read again: not
// written), 2 = fd_rhs (w <- rhs only).
template <class T, bool PATH55, int TX, int TY, int NS_, int RY, bool FORCE, int MODE>
struct Tiled {
    typedef typename Arith<T>::type A;  // arithmetic type: T itself, or V2 = two vertically adjacent fp32 cells (plain fp32)
    static constexpr int CY = Arith<T>::CY;
    static constexpr bool YP = CY == 2;   // "y pairs": T = float in memory, one thread computes cells (i, j) and (i, j+1) as one V2
    static_assert(!YP || RY == 1, "y pairs: one value (two cells) per thread");
    static constexpr bool RW = (MODE & 1) != 0, WW = (MODE & 2) != 0, WF = (MODE & 4) != 0;
    static constexpr int TH = TY * RY * CY;  // tile height in stored elements (cells, or paired-layout values)
    static constexpr int PXS = TX + 8;  // staged row: 4 values left of the tile (3 used; keeps rows 16-byte aligned) + TX + 4
    static constexpr int PYS = TH + 2 * R;
    static constexpr int FIELD = PXS * PYS;
    static constexpr int STAGE = 4 * FIELD;  // values per stage: four fields of one plane
    static constexpr int NS = NS_;           // stages (4 or 8); the plane loop is unrolled 8x, so stage offsets are immediates
    static_assert(NS == 4, "ring depth: the producer requests plane p + 3 and the w tile of the same iteration on one barrier");
    static constexpr int NW = 4;             // w stages
    static constexpr int WFIELD = TX * TH;
    static constexpr int WSTAGE = 4 * WFIELD;
    static constexpr int THREADS = TX * TY;
    static constexpr int WARPS = THREADS / 32;
    // Tensor memory as per-thread storage (8-byte value types): a warp owns the 32 lanes of its quadrant (warp % 4);
    // the warps of a quadrant use different column blocks, one per owned column.  Block = 4 delay-line slots of 16
    // columns (6 values) + 4 fields x 8 window slots of 2 columns = 128 columns.  TMEM is otherwise idle here.
    static constexpr bool TM = sizeof(A) == 8;
    static constexpr int DLCOLS = 16, TWIN = 4 * DLCOLS, TBLOCK = TWIN + 4 * 16;
    static constexpr int FXYCOL = 12;  // spare columns 12..15 of delay-line slot 0: the forcing's xy phase factors
    // when to fetch them: with the window (fp64) or after the right-hand side is assembled (paired fp32, where the
    // register pressure peaks at the window load: 144 registers and no spill instead of 168 with spills) — measured
    static constexpr bool FXY_LATE = Scalar<A>::lanes == 2;
    static constexpr int TMEM_NEED = ((WARPS + 3) / 4) * RY * TBLOCK;
    static constexpr int TMEM_COLS = TMEM_NEED <= 128 ? 128 : (TMEM_NEED <= 256 ? 256 : 512);
    static_assert(TMEM_NEED <= 512, "tensor memory has 512 columns");
    static constexpr size_t SMEM = (size_t)(NS * STAGE + NW * WSTAGE) * sizeof(T) + (2 * NS + 2) * sizeof(uint64_t);
    static size_t smem_bytes(int planes) { return SMEM + (FORCE ? 2 * (size_t)planes * sizeof(A) : 0); }  // + the z table
    static_assert((STAGE * sizeof(T)) % 128 == 0 && (WSTAGE * sizeof(T)) % 128 == 0, "TMA shared-memory boxes must stay 128-byte aligned");

    struct State {   // of one owned column
        A win[4][8];
        A lin[3][8];
        A dl[6][4];  // g_x, g_y, d_x u_z, d_y u_z, d_x u_x + d_y u_y, partial rhs_0 of the last planes (registers: !TM only)
    };

    // scatter of the in-plane differences e_m of plane t into the accumulator ring of one rhs component (Eq. 8 with z)
    template <int n8>
    static __device__ __forceinline__ void scatter(A (&lin)[8], const A (&e)[3], const KC<A>& c) {
        lin[(n8 + 3) & 7] = (-c.mq[2]) * e[2];  // first contribution to output t+3 (the sign goes with the constant: free)
        lin[(n8 + 2) & 7] = fma_(-c.mq[1], e[1], lin[(n8 + 2) & 7]);
        lin[(n8 + 1) & 7] = fma_(-c.mq[0], e[0], lin[(n8 + 1) & 7]);
        lin[(n8 + 7) & 7] = fma_(c.mq[0], e[0], lin[(n8 + 7) & 7]);
        lin[(n8 + 6) & 7] = fma_(c.mq[1], e[1], lin[(n8 + 6) & 7]);
        lin[(n8 + 5) & 7] = fma_(c.mq[2], e[2], lin[(n8 + 5) & 7]);  // output t-3 is complete
    }

    // Output plane z = t - 4, field f of one owned column: centre value, D1z and (u fields) D2z + the finished
    // accumulator, from the window ring (slot t = n8 is not among the seven used).  wr: the ring of field f as fetched
    // from tensor memory (after tcgen05.wait::ld); plain fp32: the ring is st.win[f] and slot t is rewritten with cnew.
    template <int n8>
    static __device__ __forceinline__ void zfield(int f, State& st, uint32_t (&wr)[16], A cnew, A (&fc)[4], A (&d1z)[4], A (&lz)[3], const KC<A>& c) {
        constexpr int cz = (n8 + 4) & 7;
        A w8[8];
        if constexpr (TM) {
            tmem_fence16(wr);
#pragma unroll
            for (int a8 = 0; a8 < 8; ++a8) {
                const uint2 u = make_uint2(wr[2 * a8], wr[2 * a8 + 1]);
                w8[a8] = *reinterpret_cast<const A*>(&u);
            }
        } else {
#pragma unroll
            for (int a8 = 0; a8 < 8; ++a8) w8[a8] = st.win[f][a8];
            st.win[f][n8] = cnew;  // after the read: slot t is unused by this output
        }
        const A* a = f == 0 ? c.ar : c.au;
        fc[f] = w8[cz];
        d1z[f] = fma_(a[2], w8[(cz + 3) & 7] - w8[(cz + 5) & 7], fma_(a[1], w8[(cz + 2) & 7] - w8[(cz + 6) & 7], a[0] * (w8[(cz + 1) & 7] - w8[(cz + 7) & 7])));
        if (f > 0) {
            const A* bz = f == 3 ? c.lq : c.lo;
            A v = fma_(bz[0], fc[f], st.lin[f - 1][cz]);
            v = fma_(bz[1], w8[(cz + 1) & 7] + w8[(cz + 7) & 7], v);
            v = fma_(bz[2], w8[(cz + 2) & 7] + w8[(cz + 6) & 7], v);
            v = fma_(bz[3], w8[(cz + 3) & 7] + w8[(cz + 5) & 7], v);
            lz[f - 1] = v;
        }
    }

    // ---- One iteration of the software-pipelined plane loop ---------------------------------------------------
    // In-plane work of plane t AND the output of plane z = t - 4 in ONE basic block.  The output lags the load front by
    // four planes instead of three: output z needs planes z-3 .. z+3 (all consumed in earlier iterations), so nothing
    // in the output part depends on the in-plane part of the same iteration and the compiler may interleave them:
    //   lin ring   in-plane(t) scatters into slots t-3 .. t+3; output reads slot t-4 = t+4 (mod 8): all 8 slots live
    //   window     in-plane(t) writes slot t; output reads the 7 other slots
    //   delay line slot t & 3 is read (plane t-4) BEFORE it is rewritten with the values of plane t
    //   w ring     output index q = p - 7 uses slot q & 3
    // RY == 1: the output side of field f follows the in-plane side of field f, so that its arithmetic fills the gaps
    // between the shared-memory loads of the next field (SPLIT = false).  RY > 1: the output side runs column by
    // column after the in-plane side, which keeps fewer values live at once (SPLIT = true).
    // `out` only gates the stores (warm-up iterations compute on zero-initialised state and store nothing).
    static constexpr bool SPLIT = RY > 1;
    template <int PH>
    static __device__ __forceinline__ void plane(State (&st)[RY], const T* __restrict__ sp0, const T* __restrict__ wsp0, uint32_t tdl,
                                                 const KC<A>& c, bool out, T* __restrict__ bF, T* __restrict__ bW, T* __restrict__ bD, uint32_t of, uint32_t ow,
                                                 uint32_t fs, uint32_t n, int pf, int pw, const bool (&ok)[RY], bool okb, const ForceTab<T>& ft, int ci, int cj, const A* __restrict__ ftz) {
        constexpr int n8 = PH & 7, n4 = PH & 3;
        const T* sp = sp0 + (PH & 3) * STAGE;
        const T* wsp = wsp0 + ((PH + 1) & 3) * WSTAGE;  // w ring slot of output index p - 7
        A ctr[RY][4], d1x[RY][4], d1y[RY][4], inpl[RY][3], ezx[RY][3];
        A fc[RY][4], d1z[RY][4], lz[RY][3];
        uint32_t wr[RY][16];
        if constexpr (TM && !SPLIT) {
#pragma unroll
            for (int r = 0; r < RY; ++r) tmem_ld16_nc(tdl + r * TBLOCK + TWIN, wr[r]);
        }
#pragma unroll
        for (int f = 0; f < 4; ++f) {
            // ---- plane t, field f: in-plane derivatives (Eq. 6-8).  The RY + 6 values of the thread's own x column are
            // loaded once per field and serve the y stencils of all its outputs.
            const T* q0 = sp + f * FIELD;
            A yv[YP ? 1 : RY + 2 * R];
            if constexpr (!YP) {
#pragma unroll
                for (int i = 0; i < RY + 2 * R; ++i) yv[i] = q0[(i - R) * PXS];
            }
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                const T* q = q0 + r * PXS;
                A xp1, xm1, xp2, xm2, xp3, xm3, dy1, dy2, dy3, sy1, sy2, sy3;
                if constexpr (YP) {
                    // the thread's cells are (x, a) and (x, b = a + 1), q points at (x, a).  Eight values of the x column
                    // serve both y stencils; each enters ONE packed operand (so it is loaded straight into its half of a
                    // register pair), the odd offsets are formed half by half with scalar instructions.
                    typename Scalar<A>::type cy[8];
#pragma unroll
                    for (int k = 0; k < 8; ++k) cy[k] = q[(k - R) * PXS];
                    ctr[r][f] = A(cy[3], cy[4]);
                    const A up(cy[5], cy[6]), lo(cy[1], cy[2]);  // rows a+2, b+2 and a-2, b-2
                    dy2 = up - lo;
                    dy1 = A(cy[4] - cy[2], cy[5] - cy[3]);
                    dy3 = A(cy[6] - cy[0], cy[7] - cy[1]);
                    if (f > 0) {
                        sy2 = up + lo;
                        sy1 = A(cy[4] + cy[2], cy[5] + cy[3]);
                        sy3 = A(cy[6] + cy[0], cy[7] + cy[1]);
                    }
                    xp1 = A(q[1], q[PXS + 1]); xm1 = A(q[-1], q[PXS - 1]);
                    xp2 = A(q[2], q[PXS + 2]); xm2 = A(q[-2], q[PXS - 2]);
                    xp3 = A(q[3], q[PXS + 3]); xm3 = A(q[-3], q[PXS - 3]);
                } else {
                    ctr[r][f] = yv[r + R];
                    xp1 = q[1]; xm1 = q[-1]; xp2 = q[2]; xm2 = q[-2]; xp3 = q[3]; xm3 = q[-3];
                    const A yp1 = yv[r + R + 1], ym1 = yv[r + R - 1], yp2 = yv[r + R + 2], ym2 = yv[r + R - 2], yp3 = yv[r + R + 3], ym3 = yv[r + R - 3];
                    dy1 = yp1 - ym1; dy2 = yp2 - ym2; dy3 = yp3 - ym3;
                    if (f > 0) { sy1 = yp1 + ym1; sy2 = yp2 + ym2; sy3 = yp3 + ym3; }
                }
                if constexpr (TM) {
                    const uint2 u = *reinterpret_cast<const uint2*>(&ctr[r][f]);
                    const uint32_t r2[2] = {u.x, u.y};
                    tmem_st2_nc(tdl + r * TBLOCK + TWIN + f * 16 + n8 * 2, r2);
                }
                const A dx1 = xp1 - xm1, dx2 = xp2 - xm2, dx3 = xp3 - xm3;
                const A* a = f == 0 ? c.ar : c.au;
                d1x[r][f] = fma_(a[2], dx3, fma_(a[1], dx2, a[0] * dx1));
                d1y[r][f] = fma_(a[2], dy3, fma_(a[1], dy2, a[0] * dy1));
                if (f > 0) {
                    const A sx1 = xp1 + xm1, sx2 = xp2 + xm2, sx3 = xp3 + xm3;
                    const A* bx = f == 1 ? c.lq : c.lo;  // d_xx u_x and d_yy u_y carry 4nu/3 on the 55-point path
                    const A* by = f == 2 ? c.lq : c.lo;
                    A v = c.cxy[f - 1] * ctr[r][f];
                    v = fma_(bx[1], sx1, v);
                    v = fma_(by[1], sy1, v);
                    v = fma_(bx[2], sx2, v);
                    v = fma_(by[2], sy2, v);
                    v = fma_(bx[3], sx3, v);
                    v = fma_(by[3], sy3, v);
                    if (PATH55 && (f == 1 || f == 2)) {  // Eq. 8 in the xy plane: d_xy u_x -> rhs_y, d_xy u_y -> rhs_x
                        A q1, q2, q3;
                        if constexpr (YP) {
                            // q_m = dx_m f(row + m) - dx_m f(row - m) for rows a and b.  m = 1: rows a + 1 = b and b - 1 = a
                            // are the thread's own (dx1 above), only rows a - 1 and b + 1 are loaded
                            const auto e_lo = q[-PXS + 1] - q[-PXS - 1], e_hi = q[2 * PXS + 1] - q[2 * PXS - 1];
                            q1 = A(dx1.v.y - e_lo, e_hi - dx1.v.x);
                            q2 = (A(q[2 * PXS + 2], q[3 * PXS + 2]) - A(q[2 * PXS - 2], q[3 * PXS - 2])) -
                                 (A(q[-2 * PXS + 2], q[-PXS + 2]) - A(q[-2 * PXS - 2], q[-PXS - 2]));
                            q3 = (A(q[3 * PXS + 3], q[4 * PXS + 3]) - A(q[3 * PXS - 3], q[4 * PXS - 3])) -
                                 (A(q[-3 * PXS + 3], q[-2 * PXS + 3]) - A(q[-3 * PXS - 3], q[-2 * PXS - 3]));
                        } else {
                            q1 = (q[PXS + 1] - q[PXS - 1]) + (q[-PXS - 1] - q[-PXS + 1]);
                            q2 = (q[2 * PXS + 2] - q[2 * PXS - 2]) + (q[-2 * PXS - 2] - q[-2 * PXS + 2]);
                            q3 = (q[3 * PXS + 3] - q[3 * PXS - 3]) + (q[-3 * PXS - 3] - q[-3 * PXS + 3]);
                        }
                        const A dq = fma_(c.mq[2], q3, fma_(c.mq[1], q2, c.mq[0] * q1));
                        if (f == 1) { inpl[r][0] = v; inpl[r][1] = dq; } else { inpl[r][1] += v; inpl[r][0] += dq; }
                    } else {
                        inpl[r][f - 1] = v;
                    }
                }
                if (PATH55) {  // the differences that feed Dzx u_x + Dzy u_y -> rhs_z, Dxz u_z -> rhs_x, Dyz u_z -> rhs_y
                    if (f == 1) { ezx[r][0] = dx1; ezx[r][1] = dx2; ezx[r][2] = dx3; }
                    if (f == 2) {
                        const A ez[3] = {ezx[r][0] + dy1, ezx[r][1] + dy2, ezx[r][2] + dy3};
                        scatter<n8>(st[r].lin[2], ez, c);
                    }
                    if (f == 3) {
                        const A ex[3] = {dx1, dx2, dx3}, ey[3] = {dy1, dy2, dy3};
                        scatter<n8>(st[r].lin[0], ex, c);
                        scatter<n8>(st[r].lin[1], ey, c);
                    }
                }
            }
            if constexpr (!SPLIT) {  // output side of field f right here
                if constexpr (TM) tmem_wait_ld_nc();
#pragma unroll
                for (int r = 0; r < RY; ++r) zfield<n8>(f, st[r], wr[r], ctr[r][f], fc[r], d1z[r], lz[r], c);
                if constexpr (TM) {
                    if (f < 3) {
#pragma unroll
                        for (int r = 0; r < RY; ++r) tmem_ld16_nc(tdl + r * TBLOCK + TWIN + (f + 1) * 16, wr[r]);
                    }
                }
            }
        }
        // the delayed in-plane values of plane t - 4 (slot t & 3, read before it is rewritten below)
        uint32_t dr[RY][16];
        if constexpr (TM && !SPLIT) {
#pragma unroll
            for (int r = 0; r < RY; ++r) tmem_ld16_nc(tdl + r * TBLOCK + n4 * DLCOLS, dr[r]);  // 12 values + 4 spare columns
        }
        // ---- plane t: everything of dt*rhs that needs no z derivative (Eq. 1-3); G' = dt * grad u
        A park[RY][6];
#pragma unroll
        for (int r = 0; r < RY; ++r) {
            const A gx = d1x[r][0], gy = d1y[r][0], ux = ctr[r][1], uy = ctr[r][2];
            const A Gxx = d1x[r][1], Gxy = d1y[r][1], Gyx = d1x[r][2], Gyy = d1y[r][2], Gzx = d1x[r][3], Gzy = d1y[r][3];
            const A Dh = Gxx + Gyy;
            const A ug = fma_(uy, gy, ux * gx);
            const A P0 = fma_(-c.dt, ug, -Dh);
            const A h = fma_(-c.nu23, Dh, -c.cs2dt);
            const A nsym = c.nu * (Gxy + Gyx);
            const A kx = fma_(c.nu2, Gxx, h), ky = fma_(c.nu2, Gyy, h);
            A tx = inpl[r][0], ty = inpl[r][1], tz = inpl[r][2];
            tx = fma_(-ux, Gxx, tx);
            ty = fma_(-ux, Gyx, ty);
            tx = fma_(-uy, Gxy, tx);
            ty = fma_(-uy, Gyy, ty);
            tx = fma_(gx, kx, tx);
            ty = fma_(gy, ky, ty);
            tx = fma_(nsym, gy, tx);
            ty = fma_(nsym, gx, ty);
            tz = fma_(Gzx, fma_(c.nu, gx, -ux), tz);
            tz = fma_(Gzy, fma_(c.nu, gy, -uy), tz);
            const A pl[3] = {tx, ty, tz};
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                if (PATH55)
                    st[r].lin[i][n8] += pl[i];
                else
                    st[r].lin[i][n8] = pl[i];
            }
            park[r][0] = gx; park[r][1] = gy; park[r][2] = Gzx; park[r][3] = Gzy; park[r][4] = Dh; park[r][5] = P0;
        }
        if constexpr (TM && !SPLIT) tmem_wait_ld_nc();
        // ---- output plane z = t - 4: the rest of Eq. 1-3, Eq. 10
#pragma unroll
        for (int r = 0; r < RY; ++r) {
            if constexpr (SPLIT) {  // the whole output side of this column: window rings and delay line in one batch
                uint32_t w4[4][16];
                if constexpr (TM) {
#pragma unroll
                    for (int f = 0; f < 4; ++f) tmem_ld16_nc(tdl + r * TBLOCK + TWIN + f * 16, w4[f]);
                    tmem_ld16_nc(tdl + r * TBLOCK + n4 * DLCOLS, dr[r]);
                    tmem_wait_ld_nc();
                }
#pragma unroll
                for (int f = 0; f < 4; ++f) zfield<n8>(f, st[r], w4[f], ctr[r][f], fc[r], d1z[r], lz[r], c);
            }
            A del[6];
            if constexpr (TM) {
                tmem_fence16(dr[r]);
                Regs6<A>::unpack(dr[r], del);
                uint32_t pk[12];
                Regs6<A>::pack(park[r], pk);
                tmem_st8_nc(tdl + r * TBLOCK + n4 * DLCOLS, pk);
                tmem_st4_nc(tdl + r * TBLOCK + n4 * DLCOLS + 8, pk + 8);
            } else {
#pragma unroll
                for (int q = 0; q < 6; ++q) {
                    del[q] = st[r].dl[q][n4];
                    st[r].dl[q][n4] = park[r][q];
                }
            }
            const A gxd = del[0], gyd = del[1], Gzxd = del[2], Gzyd = del[3], Dhd = del[4], P0d = del[5];
            const A gz = d1z[r][0], Gxz = d1z[r][1], Gyz = d1z[r][2], Gzz = d1z[r][3], uz = fc[r][3];
            const A divp = Dhd + Gzz;  // dt * div u
            A Rv[4];
            Rv[0] = fma_(-(c.dt * uz), gz, P0d - Gzz);
            const A ngz = c.nu * gz, m23 = c.nu23 * Gzz;
            A rx = lz[r][0], ry = lz[r][1], rz = lz[r][2];
            rx = fma_(-uz, Gxz, rx);
            ry = fma_(-uz, Gyz, ry);
            rz = fma_(-uz, Gzz, rz);
            rx = fma_(ngz, Gxz + Gzxd, rx);
            ry = fma_(ngz, Gyz + Gzyd, ry);
            rz = fma_(gz, fma_(c.nu2, Gzz, fma_(-c.nu23, divp, -c.cs2dt)), rz);
            rx = fma_(-m23, gxd, rx);
            ry = fma_(-m23, gyd, ry);
            rz = fma_(c.nu * gxd, Gxz, rz);
            rz = fma_(c.nu * gyd, Gyz, rz);
            Rv[1] = rx;
            Rv[2] = ry;
            Rv[3] = rz;
            if constexpr (FORCE) {  // + dt f_i = dt N f_k,i cos(k.x + phi), cos(a + b) = cos a cos b - sin a sin b
                A cxy = A(0), sxy = A(0);
                if constexpr (TM) {
                    if (n4 == 0) {  // the forcing's xy phase factors sit in the spare columns 12..15 of delay-line slot 0
                        const uint2 uc = make_uint2(dr[r][12], dr[r][13]), us = make_uint2(dr[r][14], dr[r][15]);
                        cxy = *reinterpret_cast<const A*>(&uc);
                        sxy = *reinterpret_cast<const A*>(&us);
                    } else {
                        uint32_t fr[4];
                        tmem_ld4_nc(tdl + r * TBLOCK + FXYCOL, fr);
                        tmem_wait_ld_nc();
                        tmem_fence4(fr);
                        const uint2 uc = make_uint2(fr[0], fr[1]), us = make_uint2(fr[2], fr[3]);
                        cxy = *reinterpret_cast<const A*>(&uc);
                        sxy = *reinterpret_cast<const A*>(&us);
                    }
                } else if (ok[r]) {
                    if constexpr (!YP) ft.xy(ci, cj + r, cxy, sxy);  // L1-resident tables: no registers held across planes
                }
                const A cth = fma_(-sxy, ftz[1], cxy * ftz[0]);
#pragma unroll
                for (int i = 0; i < 3; ++i) Rv[1 + i] = fma_(c.fa[i], cth, Rv[1 + i]);
            }
            // ---- Eq. 10; coalesced row segments per warp straight to global memory
            if (ok[r] && out) {
#pragma unroll
                for (int f = 0; f < 4; ++f) {
                    if constexpr (YP) {  // row a, and row b = a + 1 when it is inside the grid
                        A wold = A(0);
                        if (RW) wold = A(wsp[f * WFIELD], wsp[f * WFIELD + TX]);
                        const A wn = RW ? fma_(c.alpha, wold, Rv[f]) : Rv[f];
                        const A fn = fma_(c.beta, wn, fc[r][f]);
                        if (WW) bW[ow + f * n] = wn.v.x;
                        if (WF) bF[of + f * fs] = fn.v.x;
                        if (okb) {
                            if (WW) bW[ow + f * n + pw] = wn.v.y;
                            if (WF) bF[of + f * fs + pf] = fn.v.y;
                        }
                    } else {
                        const A wold = wsp[f * WFIELD + r * TX];
                        const A wn = RW ? fma_(c.alpha, wold, Rv[f]) : Rv[f];
                        if (WW) bW[ow + f * n + r * pw] = wn;
                        if (WF) bF[of + f * fs + r * pf] = fma_(c.beta, wn, fc[r][f]);
                    }
                }
                if constexpr (!PATH55) {
                    if constexpr (YP) {
                        bD[of] = divp.v.x;
                        if (okb) bD[of + pf] = divp.v.y;
                    } else {
                        bD[of + r * pf] = divp;
                    }
                }
            }
        }
    }

    static __device__ __forceinline__ void run(const Maps& m, const Geom& g, const KC<A>& c, const Sched sc, T* __restrict__ Fout,
                                               T* __restrict__ W, T* __restrict__ Div, const ForceTab<T>& ft) {
        extern __shared__ __align__(128) unsigned char smem_raw[];
        T* sm = reinterpret_cast<T*>(smem_raw);
        T* smw = sm + NS * STAGE;
        const uint32_t a_sm = __reduce_or_sync(0xffffffffu, smem_u32(smem_raw));  // uniform: kept in a uniform register
        const uint32_t a_smw = a_sm + (uint32_t)(NS * STAGE * sizeof(T));
        const uint32_t a_full = a_smw + (uint32_t)(NW * WSTAGE * sizeof(T)), a_empty = a_full + 8 * NS;
        const int tx = threadIdx.x, ty = threadIdx.y;
        const int tid = ty * TX + tx;
        const bool lane0 = (tid & 31) == 0, producer = tid == 0;
        int tile = blockIdx.x, zs = 0, ze = g.nz;
        if (sc.za > 0) {  // split list: every tile cut at plane za, the long parts first
            const int nt = sc.ntx * sc.nty;
            if (tile >= nt) {
                tile -= nt;
                zs = sc.za;
            } else {
                ze = sc.za;
            }
        } else if (tile >= sc.n_full) {
            const int j = tile - sc.n_full;
            tile = sc.n_full + j / sc.k;
            zs = (j % sc.k) * sc.zc;
            ze = min(zs + sc.zc, g.nz);
        }
        if (zs >= ze) return;  // empty chunk (rounding); the whole CTA leaves before any barrier
        const int tbx = tile % sc.ntx, tby = tile / sc.ntx;
        const int X0 = tbx * (TX - sc.ov), Y0 = tby * (TH - sc.ov);  // ov = 0 except in the temporal-blocking emulation
        const int np = ze - zs + 2 * R;  // staged planes t = zs-3 .. ze+2
        constexpr int L = Scalar<T>::lanes;
        // TMA box origin; the tensor maps count scalars along x, a value is L of them
        const int bx = (g.gx + X0 - 4) * L, by = g.gy + Y0 - R, bz = g.gz + zs - R;
        constexpr uint32_t kStageBytes = (uint32_t)(STAGE * sizeof(T));
        constexpr uint32_t kWBytes = (uint32_t)(WSTAGE * sizeof(T));
        if (producer) {
#pragma unroll
            for (int i = 0; i < NS; ++i) {
                mbar_init(a_full + 8 * i, 1);
                mbar_init(a_empty + 8 * i, WARPS);
            }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        const uint32_t a_tmem = a_empty + 8 * NS;  // shared word that receives the TMEM base address
        // FORCE: (cos, sin) of k_z z for the output planes of this item, behind the barriers
        A* ftz = reinterpret_cast<A*>(smem_raw + (size_t)(NS * STAGE + NW * WSTAGE) * sizeof(T) + (2 * NS + 2) * sizeof(uint64_t));
        if constexpr (FORCE) {
            for (int i = tid; i < ze - zs; i += THREADS) {
                T cz, sz;
                ft.z(zs + i, cz, sz);
                if constexpr (YP) { ftz[2 * i] = A(cz, cz); ftz[2 * i + 1] = A(sz, sz); } else { ftz[2 * i] = cz; ftz[2 * i + 1] = sz; }
            }
        }
        uint32_t tmem_base = 0;
        if constexpr (TM) {
            if (tid < 32) {  // warp 0 allocates (and frees) the tensor-memory columns
                asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(a_tmem), "n"(TMEM_COLS) : "memory");
                asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
            }
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            asm volatile("ld.shared.b32 %0, [%1];" : "=r"(tmem_base) : "r"(a_tmem) : "memory");
        } else {
            __syncthreads();
        }
        // a warp reaches the 32 lanes of its quadrant (warp % 4); warps that share a quadrant use different columns
        // (the address is the same for all lanes of a warp; the warp-wide OR tells the compiler so: it then lives in a
        // uniform register for the whole loop instead of being re-derived and moved there before every tcgen05 access)
        const uint32_t tdl =
            __reduce_or_sync(0xffffffffu, tmem_base + ((uint32_t)(((tid >> 5) & 3) * 32) << 16) + (uint32_t)((tid >> 7) * RY * TBLOCK));
        if (producer) {
            for (int i = 0; i < NS && i < np; ++i) {
                mbar_expect_tx(a_full + 8 * i, kStageBytes);
                tma_load_4d(a_sm + i * kStageBytes, &m.f_in, a_full + 8 * i, bx, by, bz + i, 0);
            }
        }
        const T* sp0 = sm + (ty * RY * CY + R) * PXS + (tx + 4);
        const T* wsp0 = smw + ty * RY * CY * TX + tx;
        // this thread's first cell of output plane zs in the dense (w) and padded (F, div) arrays; advanced plane by plane
        const int ci = X0 + tx, cj = Y0 + ty * RY * CY;
        bool ok[RY];
#pragma unroll
        for (int r = 0; r < RY; ++r) ok[r] = ci < g.nx && cj + r < g.ny;
        if (sc.ov > 0) {  // overlapping tiles: a value is stored by the tile whose interior (edge minus ov / 2) holds it
            const int h = sc.ov / 2;
            const bool in_x = (tbx == 0 || tx >= h) && (tbx == sc.ntx - 1 || tx < TX - h);
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                const int row = ty * RY + r;
                ok[r] = ok[r] && in_x && (tby == 0 || row >= h) && (tby == sc.nty - 1 || row < TH - h);
            }
        }
        const bool store_ok = ci < g.nx && cj < g.ny;  // the thread's first cell is inside the grid: its offsets are valid
        const bool okb = YP && ci < g.nx && cj + 1 < g.ny;  // y pairs: the second cell of the thread is inside the grid
        if constexpr (FORCE && TM) {
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                A cxy = A(0), sxy = A(0);
                if constexpr (YP) {
                    T ca = 0, sa = 0, cb = 0, sb = 0;
                    if (ok[r]) ft.xy(ci, cj, ca, sa);
                    if (okb) ft.xy(ci, cj + 1, cb, sb);
                    cxy = A(ca, cb);
                    sxy = A(sa, sb);
                } else {
                    if (ok[r]) ft.xy(ci, cj + r, cxy, sxy);
                }
                const uint2 uc = *reinterpret_cast<const uint2*>(&cxy), us = *reinterpret_cast<const uint2*>(&sxy);
                const uint32_t r4[4] = {uc.x, uc.y, us.x, us.y};
                tmem_st<4>(tdl + r * TBLOCK + FXYCOL, r4);
            }
        }
        const uint32_t plane_w = (uint32_t)g.nx * g.ny, plane_f = (uint32_t)g.px * g.py;
        // 32-bit element offsets (tiled_supported guarantees 4 fs, 4 n < 2^32): one wide multiply-add per store address
        uint32_t ow = (uint32_t)(ci + (long long)g.nx * (cj + (long long)g.ny * zs));
        uint32_t of = (uint32_t)((ci + g.gx) + (long long)g.px * ((cj + g.gy) + (long long)g.py * (zs + g.gz)));
        if (!store_ok) { ow = 0; of = 0; }
        State st[RY];
#pragma unroll
        for (int r = 0; r < RY; ++r) {
#pragma unroll
            for (int a = 0; a < 8; ++a) {
#pragma unroll
                for (int f = 0; f < 4; ++f) st[r].win[f][a] = A(0);
#pragma unroll
                for (int q = 0; q < 3; ++q) st[r].lin[q][a] = A(0);
            }
#pragma unroll
            for (int q = 0; q < 6; ++q)
#pragma unroll
                for (int a = 0; a < 4; ++a) st[r].dl[q][a] = A(0);
        }

        // Software-pipelined plane loop: iteration p stages nothing itself; it consumes plane p in-plane (p < np) and
        // finishes output index p - 7 (p >= 7), both in plane<>().  np + 1 iterations; the last one has no new plane
        // (its in-plane part re-reads a stale stage and only feeds ring slots that are never output).
        const int niter = np + 1;
        const int wid = tid >> 5;
        int pwarp = 0;  // the warp whose lane 0 requests the loads at the end of this iteration: round robin over the warps, so
                        // that no warp carries the producer's instructions and its wait for the slowest warp every iteration
        for (int pb = 0; pb < niter; pb += 8) {
#pragma unroll
            for (int ph = 0; ph < 8; ++ph) {
                const int p = pb + ph;
                if (p < niter) {
                    const bool out = p >= 2 * R + 1;
                    if constexpr (TM) tmem_wait_st_nc();  // what the previous iterations parked in tensor memory is in place
                    // ONE barrier per iteration: plane p of F and the w values of output index p - 7 were requested together
                    if (p < np || (RW && out)) mbar_wait(a_full + 8 * (ph & 3), (uint32_t)((p >> 2) & 1));
#define FD6_PLANE(K) \
    plane<K>(st, sp0, wsp0, tdl, c, out, Fout, W, Div, of, ow, (uint32_t)g.fs, (uint32_t)g.n, g.px, g.nx, ok, okb, ft, ci, cj, ftz + 2 * (p - 2 * R - 1))
                    switch (ph) {  // ph is a compile-time constant after unrolling
                        case 0: FD6_PLANE(0); break;
                        case 1: FD6_PLANE(1); break;
                        case 2: FD6_PLANE(2); break;
                        case 3: FD6_PLANE(3); break;
                        case 4: FD6_PLANE(4); break;
                        case 5: FD6_PLANE(5); break;
                        case 6: FD6_PLANE(6); break;
                        default: FD6_PLANE(7); break;
                    }
#undef FD6_PLANE
                    if (out && store_ok) {
                        ow += plane_w;
                        of += plane_f;
                    }
                    // this warp is done reading stage ph (F) and its w slot: hand them back
                    __syncwarp();
                    if (lane0) mbar_arrive(a_empty + 8 * (ph & 3));
                    // thread 0 requests what iteration q = p + 3 will consume into the stage and w slot that every warp has
                    // released one iteration earlier: plane q of F and the w values of output index q - 7, on one barrier
#ifdef FD6_FIXED_PRODUCER
                    const bool requests = producer;
#else
                    const bool requests = lane0 && wid == pwarp;
                    pwarp = pwarp + 1 == WARPS ? 0 : pwarp + 1;
#endif
                    if (requests && p >= 1) {
                        const int sq = (ph + 3) & 3;  // stage of iterations p - 1 and p + 3
                        const int q = p + 3;
                        const bool more_f = q < np;
                        const bool more_w = RW && q >= 2 * R + 1 && q < niter;
                        if (more_f || more_w) {
                            mbar_wait(a_empty + 8 * sq, (uint32_t)(((p - 1) >> 2) & 1));
                            mbar_expect_tx(a_full + 8 * sq, (more_f ? kStageBytes : 0u) + (more_w ? kWBytes : 0u));
                            if (more_f) tma_load_4d(a_sm + sq * kStageBytes, &m.f_in, a_full + 8 * sq, bx, by, bz + q, 0);
                            if (more_w) tma_load_4d(a_smw + (ph & 3) * kWBytes, &m.w_ld, a_full + 8 * sq, X0 * L, Y0, zs + q - 2 * R - 1, 0);
                        }
                    }
                }
            }
        }
        if constexpr (TM) {
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();
            if (tid < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(TMEM_COLS) : "memory");
        }
    }
};

template <class T, bool PATH55, int TX, int TY, int NS, int RY, bool FORCE, int MODE>
__global__ void __launch_bounds__(TX* TY, 1)
    k_tiled_main(const __grid_constant__ Maps m, const Geom g, const __grid_constant__ KC<typename Arith<T>::type> c, const Sched sc, T* __restrict__ Fout,
                 T* __restrict__ W, T* __restrict__ Div, const ForceTab<T> ft) {
    Tiled<T, PATH55, TX, TY, NS, RY, FORCE, MODE>::run(m, g, c, sc, Fout, W, Div, ft);
}

// ---- TiledTU<T, FORCE, S>: the instantiations of one translation unit (see fd6_tiled_host.cuh) ----------------
// fn(kernel, path55, mode) for every instantiation of the main kernel of this unit.
template <class T, bool FORCE, int S, bool P55, int MODE, class Fn>
static void each_kernel_1(Fn&& fn) {
    typedef TileShape<T, S> Sh;
    fn(&k_tiled_main<T, P55, Sh::TX, Sh::TY, Sh::NS, Sh::RY, FORCE, MODE>, P55, MODE);
}
template <class T, bool FORCE, int S, bool P55, class Fn>
static void each_kernel_2(Fn&& fn) {
    each_kernel_1<T, FORCE, S, P55, 6>(fn);  // substep 1
    each_kernel_1<T, FORCE, S, P55, 7>(fn);  // substep 2
    each_kernel_1<T, FORCE, S, P55, 5>(fn);  // substep 3
    each_kernel_1<T, FORCE, S, P55, 2>(fn);  // fd_rhs
}
template <class T, bool FORCE, int S, class Fn>
static void for_each_kernel(Fn&& fn) {
    each_kernel_2<T, FORCE, S, true>(fn);
    each_kernel_2<T, FORCE, S, false>(fn);
}

template <class T, bool FORCE, int S>
size_t TiledTU<T, FORCE, S>::smem_bytes(int planes) {  // the same for every instantiation of the unit
    typedef TileShape<T, S> Sh;
    return Tiled<T, true, Sh::TX, Sh::TY, Sh::NS, Sh::RY, FORCE, 7>::smem_bytes(planes);
}
template <class T, bool FORCE, int S>
cudaError_t TiledTU<T, FORCE, S>::set_smem(size_t bytes) {
    cudaError_t e = cudaSuccess;
    for_each_kernel<T, FORCE, S>([&](auto kernel, bool, int) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    });
    return e;
}
template <class T, bool FORCE, int S>
int TiledTU<T, FORCE, S>::max_ctas_per_sm(size_t bytes) {
    typedef TileShape<T, S> Sh;
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_tiled_main<T, true, Sh::TX, Sh::TY, Sh::NS, Sh::RY, FORCE, 7>, Sh::TX * Sh::TY, bytes) !=
        cudaSuccess) {
        cudaGetLastError();
        return -1;
    }
    return n;
}
template <class T, bool FORCE, int S>
bool TiledTU<T, FORCE, S>::launch(bool path55, int mode, int items, size_t smem, cudaStream_t stream, const Maps& m, const Geom& g,
                                  const KC<typename Arith<T>::type>& c, const Sched& sc, T* Fout, T* W, T* Div, const ForceTab<T>& ft) {
    dim3 block(TileShape<T, S>::TX, TileShape<T, S>::TY, 1), grid(items, 1, 1);
    bool launched = false;
    for_each_kernel<T, FORCE, S>([&](auto kernel, bool k55, int kmode) {
        if (!launched && k55 == path55 && kmode == mode) {
            kernel<<<grid, block, smem, stream>>>(m, g, c, sc, Fout, W, Div, ft);
            launched = true;
        }
    });
    return launched;
}

}  // namespace fd6
