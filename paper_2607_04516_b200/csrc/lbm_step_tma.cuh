// lbm_step_tma.cuh — the production stream-collide kernel (a5/a6 of SURVEY.md §8) for sm_100a:
// persistent CTAs, bulk-async (TMA engine, cp.async.bulk) tile loads into a multi-stage shared-memory ring
// signalled by mbarriers, one cell per thread out of shared memory, coalesced direct stores.
//
// Why this shape (ncu, profiles/r01_step_v1_ncu.md): the one-cell-per-thread LDG kernel moves exactly the algorithmic
// bytes but issues ~650 warp instructions per cell, 200 of them 64-bit address arithmetic, and keeps only ~25 warps of
// loads in flight per SM: 60 % of DRAM peak at 57 % issue utilisation.  Here a tile of T consecutive cells of the
// linear [z][y][x] index needs, for direction i, the contiguous range [c0 - off_i, c0 - off_i + T) of population i
// (off_i = cx + cy nx + cz nx ny): ONE bulk copy per direction per tile, issued by one lane each, no per-thread
// address arithmetic, and S-1 tiles (~20 KB each) in flight per CTA independent of occupancy and registers.
// Bulk copies need 16-byte aligned addresses: the copy starts at the aligned-down element and the consumer reads at
// a per-direction shift (0..3 elements), which in shared memory is free.  Cells on domain faces or next to solids
// were loaded "as if interior"; they repair the affected directions from global memory (rare, L2-resident).
#pragma once
#include "lbm_kernels.cuh"

namespace lbmk {

// per-launch table: for direction i, src_off[i] = i*stride - off_i - shift[i]  (elements; multiple of 16/sizeof(real))
struct TmaTab {
    long long src_off[Q];
    int shift[Q];
    int bytes[Q]; // bytes of one row copy: (T + (shift ? VE : 0)) * sizeof(real)
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// global -> shared bulk copy, completion counted in bytes on the mbarrier
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
}

template <typename real, int T>
struct TmaCfg {
    static constexpr int VE = 16 / (int)sizeof(real);        // elements per 16 bytes
    static constexpr int PW = T + VE;                        // row pitch in elements (16-byte multiple)
    static constexpr int ROWS_BYTES = Q * PW * (int)sizeof(real);
    static constexpr int STAGE_BYTES = ROWS_BYTES + T;       // + T flag bytes (T % 16 == 0)
    static constexpr size_t smem_bytes(int stages) { return (size_t)stages * STAGE_BYTES + (size_t)stages * 8 + 16; }
};

// shift of direction I inside its shared-memory row when nx and nx*ny are multiples of VE (compile time)
template <int I, int VE>
__host__ __device__ constexpr int aligned_shift() { return ((-dir_cx(I)) % VE + VE) % VE; }

// T = cells per tile = threads per CTA; S = ring stages; MINB = CTAs per SM the register budget is held to.
template <typename real, bool MEAN, bool ALIGNED, int T, int S, int MINB>
__global__ void __launch_bounds__(T, MINB)
step_tma_kernel(const real *__restrict__ A, real *__restrict__ B, const uint8_t *__restrict__ flags, real *__restrict__ msum,
                const Params<real> P, const TmaTab tab, const int ntiles, const uint32_t tile_bytes)
{
    using C = TmaCfg<real, T>;
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const bool issuer = tid < 32; // warp 0 issues the bulk copies, one row per lane
    const uint32_t smem0 = smem_u32(smem);
    const uint32_t bar0 = smem0 + (uint32_t)(S * C::STAGE_BYTES);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < S; ++s) mbar_init(bar0 + 8u * s, 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    // one lane per row: rows 0..18 = populations, row 19 = the tile's flag bytes
    const real *my_src = nullptr;
    uint32_t my_dst = 0, my_bytes = 0;
    if (issuer) {
        if (lane < Q) {
            my_src = A + tab.src_off[lane];
            my_dst = (uint32_t)(lane * C::PW * (int)sizeof(real));
            my_bytes = (uint32_t)tab.bytes[lane];
        } else if (lane == Q) {
            my_dst = (uint32_t)C::ROWS_BYTES;
            my_bytes = (uint32_t)T;
        }
    }
    auto issue = [&](int tile, int s) {
        const uint32_t bar = bar0 + 8u * s;
        const uint32_t stage = smem0 + (uint32_t)(s * C::STAGE_BYTES);
        const long long c0 = (long long)tile * T;
        if (lane == 0) mbar_expect_tx(bar, tile_bytes);
        __syncwarp();
        if (lane < Q) bulk_g2s(stage + my_dst, my_src + c0, my_bytes, bar);
        else if (lane == Q) bulk_g2s(stage + my_dst, flags + c0, my_bytes, bar);
    };

    if (issuer) {
#pragma unroll
        for (int j = 0; j < S; ++j) {
            const int tile = blockIdx.x + j * gridDim.x;
            if (tile < ntiles) issue(tile, j);
        }
    }

    int s = 0;
    uint32_t parity = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const unsigned char *stage = smem + s * C::STAGE_BYTES;
        const real *rows = reinterpret_cast<const real *>(stage) + tid;
        mbar_wait(bar0 + 8u * s, parity);
        real g[Q];
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            if constexpr (ALIGNED) g[i] = rows[i * C::PW + aligned_shift<i, C::VE>()];
            else g[i] = rows[i * C::PW + tab.shift[i]];
        });
        const uint8_t fl = stage[C::ROWS_BYTES + tid];
        __syncthreads(); // every thread holds its cell in registers: the stage can be refilled
        if (issuer) {
            const int nt = tile + S * gridDim.x;
            if (nt < ntiles) issue(nt, s);
        }
        if (++s == S) { s = 0; parity ^= 1u; }

        const long long cell_ll = (long long)tile * T + tid;
        if (cell_ll >= P.N) continue;
        const int cell = (int)cell_ll;
        const int cls = fl & CLASS_MASK;
        if (cls == SOLID) continue;
        Macro<real> m;
        if (cls == EQ_FIXED) {
            if constexpr (MEAN) {
                load_cell(g, A, P.stride, cell);
                m = local_macros(g, EQ_FIXED, P);
                msum[cell] += m.ux;
                msum[P.stride + cell] += m.uy;
                msum[2 * P.stride + cell] += m.uz;
            }
            continue;
        }
        if (cls == EQ_OUTFLOW) {
            const int x = cell % P.nx, y = (cell / P.nx) % P.ny, z = cell / P.nxy;
            const int nb = outflow_neighbour(P, x, y, z);
            m = Macro<real>{real(1), real(0), real(0), real(0)};
            if (nb >= 0) {
                load_cell(g, A, P.stride, nb);
                m = local_macros(g, flags[nb] & CLASS_MASK, P);
            }
            equilibrium(g, real(0), m.ux, m.uy, m.uz);
        } else {
            if (fl & EDGE_BIT) {
                // cell on a domain face: periodic wrap / free-slip mirror / wall, then solidity of the resolved source
                const int x = cell % P.nx, y = (cell / P.nx) % P.ny, z = cell / P.nxy;
                const uint32_t bb = link_mask_edge(P, flags, x, y, z);
                g[0] = A[cell];
                static_for<1, Q>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    int sc, j;
                    resolve_geom<i>(P, x, y, z, sc, j);
                    const bool b = (bb >> i) & 1u;
                    g[i] = A[(long long)(b ? dir_opp(i) : j) * P.stride + (b ? cell : sc)];
                });
            } else if (fl & SLOW_BIT) {
                // interior cell next to a solid: bounce-back links take the cell's own opposite population
                const uint32_t bb = link_mask_interior(P, flags, cell);
                static_for<1, Q>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    if ((bb >> i) & 1u) g[i] = A[(long long)dir_opp(i) * P.stride + cell];
                });
            }
            m = collide(g, P);
        }
        real *b = B + cell;
#pragma unroll
        for (int i = 0; i < Q; ++i) b[(long long)i * P.stride] = g[i];
        if constexpr (MEAN) {
            msum[cell] += m.ux;
            msum[P.stride + cell] += m.uy;
            msum[2 * P.stride + cell] += m.uz;
        }
    }
}

// host: the per-launch table
template <typename real>
inline TmaTab make_tma_tab(const Params<real> &P, int T, uint32_t *tile_bytes, bool *aligned)
{
    constexpr int VE = 16 / (int)sizeof(real);
    TmaTab t{};
    uint32_t total = (uint32_t)T;
    for (int i = 0; i < Q; ++i) {
        const long long off = dir_cx(i) + (long long)dir_cy(i) * P.nx + (long long)dir_cz(i) * P.nxy;
        const int shift = (int)(((-off) % VE + VE) % VE);
        t.shift[i] = shift;
        t.src_off[i] = (long long)i * P.stride - off - shift;
        t.bytes[i] = (T + (shift ? VE : 0)) * (int)sizeof(real);
        total += (uint32_t)t.bytes[i];
    }
    *tile_bytes = total;
    *aligned = (P.nx % VE == 0) && (P.nxy % VE == 0);
    return t;
}

} // namespace lbmk
