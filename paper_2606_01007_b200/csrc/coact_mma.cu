// S1+S2 tensor path (TACG_PATH_MMA): C_f = X_f^T X_f over the 0/1 token x expert multi-hot matrix
// of each family (PAPER.md:71 restated as a contraction; north_star), exact in kind::i8 with s32
// accumulators.  The diagonal of X_f^T X_f is D[f,:].
//
// coact_mma_kernel, persistent, one CTA per SM, 16 producer warps + 1 MMA warp:
//   producers  load token rows (prefetched one item ahead), bin the tokens of an item by family
//              (warp ballots + one shared atomic per warp and family), expand each token's ids to a
//              row of Epad bytes in registers (bit mask -> bytes) and store it with 16-byte stores
//              into a K-chunk of its family: 32 token rows in the MN-major no-swizzle canonical
//              layout [Epad/16][32 rows][16 bytes].  Unused rows of a family's last chunk are zeroed.
//   MMA warp   one lane issues, per chunk, tcgen05.mma kind::i8 with the SAME shared-memory tile as
//              A and B (both MN-major): D_f[Epad x Epad] += X^T X in TMEM (F * Epad columns).
//   Two operand buffers alternate (full/empty mbarriers); at the end of each (CTA, layer) visit
//   warps 0-3 read the accumulators with tcgen05.ld and write them to a scratch slot.
// coact_mma_finalize_kernel sums the slots of a layer into C (off-diagonal) and D (diagonal).
//
// Dense work is Epad^2 MACs per token where the method needs k(k-1)/2 increments: bench.py
// reports the useful/dense ratio beside any tensor-pipe figure.
#include "tacg_common.cuh"
#include "umma.cuh"

namespace {

constexpr int kProducers = 512;                 // 16 warps
constexpr int kMmaThreads = kProducers + 32;    // + the MMA warp
constexpr int kMaxF = 8;

struct MmaParams {
    const int16_t* indices;
    const int8_t* family;
    long long N;
    int k, L, E, F;
    int cps;            // items per layer
    long long T;        // L * cps
    int groups;
    int nfg;            // 1: a CTA accumulates all F families; F: CTA c accumulates family c % F only
    int Fl;             // families per CTA (F or 1)
    unsigned* scratch;  // [(groups+L-1)*nfg][slot_words]
    int slot_words;     // Fl*E*E + Fl, rounded up to 4
};

template <int EP>
struct MmaGeom {
    static constexpr int kItem = EP == 64 ? 1024 : (EP == 128 ? 512 : 256);   // tokens scanned per item
    static constexpr int kTPT = kItem >= kProducers ? kItem / kProducers : 1;  // tokens per producer thread
    static constexpr int kMaxFam = EP == 64 ? 8 : (EP == 128 ? 4 : 1);         // families per CTA (TMEM columns)
    static constexpr int kTile = EP < 128 ? EP : 128;             // M = N of one tcgen05.mma
    static constexpr int kTiles = EP == 256 ? 3 : 1;              // EP = 256: tiles (0,0), (0,1), (1,1) of the symmetric product
    static constexpr int kChunks = kItem / 32 + kMaxFam;          // worst case chunks per item
    static constexpr int kChunkBytes = EP * 32;                   // [EP/16][32][16]
    static constexpr int kBufBytes = (kChunks + 1) * kChunkBytes; // + one all-zero chunk
};

__device__ __forceinline__ void producer_barrier() { asm volatile("bar.sync 1, %0;" ::"n"(kProducers) : "memory"); }

// 4 mask bits (nibble) -> 4 bytes of 0/1
__device__ __forceinline__ unsigned nibble_to_bytes(unsigned nib) { return (nib * 0x00204081u) & 0x01010101u; }

// Writes one token row (mask = EP bits) at row kk of the chunk at `chunk` (shared-space address).
template <int EP>
__device__ __forceinline__ void store_row(uint32_t chunk, int kk, const unsigned (&mask)[EP / 32]) {
#pragma unroll
    for (int c = 0; c < EP / 16; ++c) {
        const unsigned bits = (mask[c >> 1] >> ((c & 1) * 16)) & 0xffffu;
        const unsigned w0 = nibble_to_bytes(bits & 0xfu);
        const unsigned w1 = nibble_to_bytes((bits >> 4) & 0xfu);
        const unsigned w2 = nibble_to_bytes((bits >> 8) & 0xfu);
        const unsigned w3 = nibble_to_bytes(bits >> 12);
        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(chunk + c * 512 + kk * 16), "r"(w0), "r"(w1),
                     "r"(w2), "r"(w3)
                     : "memory");
    }
}

template <int EP>
__device__ __forceinline__ void zero_row(uint32_t chunk, int kk) {
#pragma unroll
    for (int c = 0; c < EP / 16; ++c)
        asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(chunk + c * 512 + kk * 16), "r"(0u) : "memory");
}

template <int KT>
__device__ __forceinline__ void load_words(const int16_t* __restrict__ row, unsigned (&w)[KT / 2]) {
    if constexpr (KT == 8) {
        const uint4 v = __ldg(reinterpret_cast<const uint4*>(row));
        w[0] = v.x; w[1] = v.y; w[2] = v.z; w[3] = v.w;
    } else if constexpr (KT == 4) {
        const uint2 v = __ldg(reinterpret_cast<const uint2*>(row));
        w[0] = v.x; w[1] = v.y;
    } else {
#pragma unroll
        for (int i = 0; i < KT / 2; ++i) w[i] = __ldg(reinterpret_cast<const unsigned*>(row) + i);
    }
}

// ids -> bit mask; ids outside [0,E) are empty slots; a duplicate id sets its bit once
template <int EP, int KT>
__device__ __forceinline__ void ids_to_mask(const unsigned (&w)[KT / 2], int E, unsigned (&mask)[EP / 32]) {
#pragma unroll
    for (int i = 0; i < EP / 32; ++i) mask[i] = 0u;
#pragma unroll
    for (int j = 0; j < KT; ++j) {
        const int e = (j & 1) ? ((int)w[j >> 1] >> 16) : (int)(short)(w[j >> 1] & 0xffffu);
        const unsigned bit = ((unsigned)e < (unsigned)E) ? (1u << (e & 31)) : 0u;
#pragma unroll
        for (int i = 0; i < EP / 32; ++i) mask[i] |= ((e >> 5) == i) ? bit : 0u;
    }
}

template <int EP, int KT>
__global__ void __launch_bounds__(kMmaThreads, 1) coact_mma_kernel(const MmaParams p) {
    tacg_pdl_prologue();
    using G = MmaGeom<EP>;
    extern __shared__ __align__(128) unsigned char opbuf[];      // [2][kChunks + 1][kChunkBytes]
    __shared__ uint64_t full_bar[2], empty_bar[2], tmem_free_bar;
    __shared__ unsigned cnt[2][kMaxF];
    __shared__ unsigned ntok_acc[kMaxF];
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = blockIdx.x / p.nfg;
    const int fsel = blockIdx.x % p.nfg;      // filter mode (nfg > 1): the one family this CTA accumulates
    const long long lo = group_lo(g, p.T, p.groups), hi = group_lo(g + 1, p.T, p.groups);
    const int F = p.Fl, E = p.E;              // F = families accumulated by this CTA
    constexpr uint32_t kTmemCols = 512;       // F * EP <= 512; one CTA per SM owns all of TMEM

    if (tid == 0) {
        umma::mbar_init(&full_bar[0], kProducers);
        umma::mbar_init(&full_bar[1], kProducers);
        umma::mbar_init(&empty_bar[0], 2);      // tcgen05.commit + the MMA thread's own arrive
        umma::mbar_init(&empty_bar[1], 2);
        umma::mbar_init(&tmem_free_bar, 128);   // warps 0-3 after draining TMEM
        umma::fence_barrier_init();
    }
    if (tid < 2 * kMaxF) cnt[tid / kMaxF][tid % kMaxF] = 0u;
    if (tid < kMaxF) ntok_acc[tid] = 0u;
    // the all-zero chunk at the end of each buffer
    for (int i = tid; i < 2 * G::kChunkBytes / 16; i += kMmaThreads) {
        const int b = i / (G::kChunkBytes / 16), o = i % (G::kChunkBytes / 16);
        reinterpret_cast<uint4*>(opbuf + (size_t)b * G::kBufBytes + (size_t)G::kChunks * G::kChunkBytes)[o] =
            make_uint4(0u, 0u, 0u, 0u);
    }
    if (warp == 0) umma::tmem_alloc(&tmem_base_s, kTmemCols);
    umma::fence_proxy_async();
    umma::tc_fence_before();
    __syncthreads();
    umma::tc_fence_after();
    const uint32_t tmem = tmem_base_s;
    const uint32_t buf0 = umma::smem_u32(opbuf);
    const long long nitems = hi - lo;

    if (warp < kProducers / 32) {
        // ================================ producers ================================
        int fam[2][G::kTPT];
        unsigned w[2][G::kTPT][KT / 2];
        auto load_item = [&](long long item, int slot) {
            const int l = (int)(item / p.cps);
            const long long t0 = (item - (long long)l * p.cps) * G::kItem;
            const int16_t* lbase = p.indices + (size_t)l * (size_t)p.N * KT;
#pragma unroll
            for (int u = 0; u < G::kTPT; ++u) {
                const int ot = tid + u * kProducers;
                const long long t = t0 + ot;
                fam[slot][u] = -1;
                if (ot < G::kItem && t < p.N) {
                    int f = p.family[t];
                    if (p.nfg > 1) f = (f == fsel) ? 0 : -1;        // filter mode: local family 0 or skipped
                    fam[slot][u] = f;
                    if (f >= 0) load_words<KT>(lbase + (size_t)t * KT, w[slot][u]);
                }
            }
        };
        if (nitems > 0) load_item(lo, 0);
        int layer = nitems > 0 ? (int)(lo / p.cps) : 0;
        int ci = (int)(lo - (long long)layer * p.cps);
#pragma unroll 1
        for (long long it = 0; it < nitems; ++it) {
            const int cur = (int)(it & 1);            // register slot and operand buffer of this item
            if (it + 1 < nitems) {                     // prefetch the next item's rows
                if (cur == 0) load_item(lo + it + 1, 1); else load_item(lo + it + 1, 0);
            }
            const uint32_t use = (uint32_t)(it >> 1);
            umma::mbar_wait(&empty_bar[cur], (use & 1u) ^ 1u);     // MMAs that read this buffer two items ago are done
            // phase A: position of each token inside its family
            int pos[G::kTPT];
#pragma unroll
            for (int u = 0; u < G::kTPT; ++u) {
                const int f = cur == 0 ? fam[0][u] : fam[1][u];
                pos[u] = -1;
#pragma unroll
                for (int q = 0; q < kMaxF; ++q) {
                    if (q < F) {
                        const unsigned m = __ballot_sync(0xffffffffu, f == q);
                        unsigned base = 0;
                        if (lane == 0 && m) base = atomicAdd(&cnt[cur][q], (unsigned)__popc(m));
                        base = __shfl_sync(0xffffffffu, base, 0);
                        if (f == q) pos[u] = (int)(base + __popc(m & ((1u << lane) - 1u)));
                    }
                }
            }
            producer_barrier();
            // phase B: chunk offsets of the families, then the rows
            unsigned n[kMaxF], off[kMaxF];
            unsigned run = 0;
#pragma unroll
            for (int q = 0; q < kMaxF; ++q) {
                n[q] = q < F ? cnt[cur][q] : 0u;
                off[q] = run;
                run += (n[q] + 31u) >> 5;
            }
            const uint32_t buf = buf0 + (uint32_t)cur * G::kBufBytes;
#pragma unroll
            for (int u = 0; u < G::kTPT; ++u) {
                const int f = cur == 0 ? fam[0][u] : fam[1][u];
                if (pos[u] >= 0) {
                    unsigned mask[EP / 32];
                    if (cur == 0) ids_to_mask<EP, KT>(w[0][u], E, mask); else ids_to_mask<EP, KT>(w[1][u], E, mask);
                    unsigned o = 0;
#pragma unroll
                    for (int q = 0; q < kMaxF; ++q) o = (f == q) ? off[q] : o;
                    store_row<EP>(buf + (o + ((unsigned)pos[u] >> 5)) * G::kChunkBytes, pos[u] & 31, mask);
                }
            }
            if (tid < F * 32) {                        // zero the unused rows of each family's last chunk
                const int q = tid >> 5;
                unsigned nq = 0, oq = 0;
#pragma unroll
                for (int z = 0; z < kMaxF; ++z) { nq = (q == z) ? n[z] : nq; oq = (q == z) ? off[z] : oq; }
                if ((nq & 31u) != 0u && (unsigned)lane >= (nq & 31u))
                    zero_row<EP>(buf + (oq + (nq >> 5)) * G::kChunkBytes, lane);
            }
            if (layer == 0 && tid < F) ntok_acc[tid] += cnt[cur][tid];
            umma::fence_proxy_async();
            umma::mbar_arrive(&full_bar[cur]);
            // end of this (CTA, layer) visit: drain the accumulators into the scratch slot
            ++ci;
            const bool last_of_visit = (ci == p.cps) || (it + 1 == nitems);
            if (last_of_visit) {
                if (warp < 4) {
                    umma::mbar_wait(&empty_bar[cur], use & 1u);     // every MMA issued so far has completed
                    umma::tc_fence_after();
                    unsigned* slot = p.scratch + ((size_t)(g + layer) * p.nfg + fsel) * p.slot_words;
                    const int lrow = EP == 64 ? warp * 16 + lane : warp * 32 + lane;   // row inside a tile
                    const bool lane_ok = EP != 64 || lane < 16;                       // M = 64: lanes 0-15 of a sub-partition
                    for (int f = 0; f < F; ++f) {
#pragma unroll
                        for (int tile = 0; tile < G::kTiles; ++tile) {
                            const int mi = tile == 2 ? 1 : 0, ni = tile == 0 ? 0 : 1;
                            const int row = mi * 128 + lrow;
                            const bool row_ok = lane_ok && row < E;
                            for (int col = 0; col < G::kTile && ni * 128 + col < E; col += 16) {
                                uint32_t v[16];
                                umma::tmem_ld_32x32b_x16(tmem + ((uint32_t)(warp * 32) << 16) +
                                                             (uint32_t)(f * EP + tile * 128 * (EP == 256) + col), v);
                                umma::tmem_ld_wait();
                                if (row_ok) {
                                    unsigned* dst = slot + ((size_t)f * E + row) * E + ni * 128 + col;
#pragma unroll
                                    for (int j = 0; j < 16; ++j)
                                        if (ni * 128 + col + j < E) dst[j] = v[j];
                                }
                            }
                        }
                    }
                    if (tid < F) {
                        slot[(size_t)F * E * E + tid] = ntok_acc[tid];
                        ntok_acc[tid] = 0u;
                    }
                    umma::tc_fence_before();
                    umma::mbar_arrive(&tmem_free_bar);
                }
                if (ci == p.cps) { ci = 0; ++layer; }
            }
        }
    } else {
        // ================================ MMA warp ================================
        const uint32_t idesc = umma::idesc_u8_mn(G::kTile, G::kTile);
        int ci = nitems > 0 ? (int)(lo - (lo / p.cps) * p.cps) : 0;
        bool first = true;            // first item of a (CTA, layer) visit: accumulators start from zero
        uint32_t visits = 0;
        unsigned accmask = 0u;        // families whose accumulator has been written in this visit
#pragma unroll 1
        for (long long it = 0; it < nitems; ++it) {
            const int cur = (int)(it & 1);
            const uint32_t use = (uint32_t)(it >> 1);
            umma::mbar_wait(&full_bar[cur], use & 1u);
            umma::tc_fence_after();
            unsigned n[kMaxF];
#pragma unroll
            for (int q = 0; q < kMaxF; ++q) n[q] = q < F ? cnt[cur][q] : 0u;
            __syncwarp();
            if (lane < kMaxF) cnt[cur][lane] = 0u;          // ready for the item after next
            __syncwarp();
            if (first) {
                if (visits > 0) umma::mbar_wait(&tmem_free_bar, (visits - 1u) & 1u);   // the previous visit was drained
                umma::tc_fence_after();
                accmask = 0u;
                ++visits;
            }
            if (lane == 0) {
                const uint32_t buf = buf0 + (uint32_t)cur * G::kBufBytes;
                unsigned off = 0;
#pragma unroll
                for (int q = 0; q < kMaxF; ++q) {
                    if (q < F) {
                        const unsigned nch = (n[q] + 31u) >> 5;
                        // chunk c == nch is the all-zero chunk: it clears the accumulators of a family that has no token yet
                        const unsigned nrun = (first && nch == 0) ? 1u : nch;
                        for (unsigned c = 0; c < nrun; ++c) {
                            const uint32_t chunk = buf + (nch ? off + c : (unsigned)G::kChunks) * G::kChunkBytes;
#pragma unroll
                            for (int tile = 0; tile < G::kTiles; ++tile) {
                                const int mi = tile == 2 ? 1 : 0, ni = tile == 0 ? 0 : 1;
                                // a tile's 128 experts are 8 column blocks of 512 bytes
                                const uint64_t da = umma::smem_desc_mn_interleave(chunk + mi * 4096 * (EP == 256), 128, 512);
                                const uint64_t db = umma::smem_desc_mn_interleave(chunk + ni * 4096 * (EP == 256), 128, 512);
                                umma::mma_i8_ss(tmem + (uint32_t)(q * EP + tile * 128 * (EP == 256)), da, db, idesc,
                                                (accmask >> q) & 1u);
                            }
                            accmask |= 1u << q;
                        }
                        off += nch;
                    }
                }
                umma::mma_commit(&empty_bar[cur]);
                __threadfence_block();
                umma::mbar_arrive(&empty_bar[cur]);
            }
            accmask = __shfl_sync(0xffffffffu, accmask, 0);
            __syncwarp();
            ++ci;
            first = false;
            if (ci == p.cps) { ci = 0; first = true; }
        }
    }
    umma::tc_fence_before();
    __syncthreads();
    if (warp == 0) umma::tmem_dealloc(tmem, kTmemCols);
}

// One CTA per (layer, family): C (off-diagonal) and D (diagonal) from the slots of the layer.
template <bool ZERO>
__global__ void __launch_bounds__(512) coact_mma_finalize_kernel(const MmaParams p, unsigned* __restrict__ D,
                                                                unsigned* __restrict__ C,
                                                                unsigned long long* __restrict__ ntok) {
    tacg_pdl_prologue();
    const int l = blockIdx.x / p.F, f = blockIdx.x % p.F;
    const int E = p.E;
    const int g0 = group_of_item((long long)l * p.cps, p.T, p.groups);
    const int g1 = group_of_item((long long)(l + 1) * p.cps - 1, p.T, p.groups);
    const int ng = g1 - g0 + 1;
    const int fgi = p.nfg > 1 ? f : 0;                   // which CTA of a group holds family f
    const int fs = p.nfg > 1 ? 0 : f;                    // family index inside a slot
    const unsigned* slot0 = p.scratch + ((size_t)(g0 + l) * p.nfg + fgi) * p.slot_words;
    const size_t gs = (size_t)p.nfg * p.slot_words;
    unsigned* Cf = C + ((size_t)l * p.F + f) * E * E;
    unsigned* Df = D + ((size_t)l * p.F + f) * E;
    for (int idx = threadIdx.x; idx < E * E; idx += blockDim.x) {
        // E > 128: the (rows >= 128, columns < 128) block is not computed; read its mirror image
        const int ii = idx / E, jj = idx - ii * E;
        const int sidx = (ii >= 128 && jj < 128) ? jj * E + ii : idx;
        const unsigned* src = slot0 + (size_t)fs * E * E + sidx;
        unsigned a0 = 0, a1 = 0;
        int g = 0;
        for (; g + 2 <= ng; g += 2) {
            a0 += src[(size_t)g * gs];
            a1 += src[(size_t)(g + 1) * gs];
        }
        if (g < ng) a0 += src[(size_t)g * gs];
        const unsigned v = a0 + a1;
        const int i = idx / E, j = idx - i * E;
        if (i == j) {
            Df[i] = ZERO ? v : Df[i] + v;
            if (ZERO) Cf[idx] = 0u;
        } else {
            Cf[idx] = ZERO ? v : Cf[idx] + v;
        }
    }
    if (l == 0 && threadIdx.x == 0) {
        unsigned long long acc = 0;
        for (int g = 0; g < ng; ++g) acc += slot0[(size_t)g * gs + (size_t)p.Fl * E * E + fs];
        ntok[f] = ZERO ? acc : ntok[f] + acc;
    }
}

template <int EP, int KT>
int launch_mma(tacg_ctx* ctx, const MmaParams& p) {
    using G = MmaGeom<EP>;
    const size_t smem = 2 * (size_t)G::kBufBytes;
    auto kern = coact_mma_kernel<EP, KT>;
    TACG_CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    TACG_CUDA_TRY(ctx, tacg_launch_pdl(kern, dim3(p.groups * p.nfg), dim3(kMmaThreads), smem, ctx->stream, p));
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}

template <int EP>
int launch_mma_k(tacg_ctx* ctx, const MmaParams& p) {
    switch (p.k) {
        case 2: return launch_mma<EP, 2>(ctx, p);
        case 4: return launch_mma<EP, 4>(ctx, p);
        case 6: return launch_mma<EP, 6>(ctx, p);
        default: return launch_mma<EP, 8>(ctx, p);
    }
}

int padded_E(int E) { return E <= 64 ? 64 : (E <= 128 ? 128 : 256); }

}  // namespace

// k even and <= 8 (vector row loads), E <= 256.  All F families share a CTA when F * Epad <= 512 TMEM
// columns and Epad <= 128; otherwise each CTA accumulates one family (Epad = 256: three 128 x 128
// tiles of the symmetric product).  The caller also checks the 16-byte alignment of `indices`.
bool tacg_coact_mma_supported(int k, int E, int F) {
    if (!(k == 2 || k == 4 || k == 6 || k == 8)) return false;
    return E >= 1 && E <= 256 && F >= 1;
}

int tacg_launch_coact_mma(tacg_ctx* ctx, const int16_t* indices, const int8_t* family, int64_t N, int k, int L,
                          int E, int F, uint32_t* D, uint32_t* C, uint64_t* ntok, bool zero_first) {
    if (!tacg_coact_mma_supported(k, E, F)) {
        snprintf(ctx->detail, sizeof(ctx->detail), "coact: shape not supported by the tcgen05 path");
        return TACG_ERR_SHAPE;
    }
    const int EP = padded_E(E);
    MmaParams p;
    p.indices = indices; p.family = family; p.N = N; p.k = k; p.L = L; p.E = E; p.F = F;
    const int item = EP == 64 ? MmaGeom<64>::kItem : (EP == 128 ? MmaGeom<128>::kItem : MmaGeom<256>::kItem);
    const bool filter = EP == 256 || F * EP > 512;
    p.nfg = filter ? F : 1;
    p.Fl = filter ? 1 : F;
    p.cps = (int)((N + item - 1) / item);
    p.T = (long long)L * p.cps;
    p.groups = (int)max(1ll, min((long long)(ctx->sm_count / p.nfg), p.T));
    p.slot_words = (int)tacg_align_up((size_t)p.Fl * E * E + p.Fl, 4);
    const size_t slots = ((size_t)p.groups + L - 1) * p.nfg;
    p.scratch = static_cast<unsigned*>(tacg_scratch(ctx, slots * p.slot_words * sizeof(unsigned)));
    if (!p.scratch) return TACG_ERR_CUDA;
    tacg_prof_scope prof(ctx, TACG_PROF_COACT);
    int rc = EP == 64 ? launch_mma_k<64>(ctx, p) : (EP == 128 ? launch_mma_k<128>(ctx, p) : launch_mma_k<256>(ctx, p));
    if (rc != TACG_OK) return rc;
    unsigned long long* nt = reinterpret_cast<unsigned long long*>(ntok);
    if (zero_first) TACG_CUDA_TRY(ctx, tacg_launch_pdl(coact_mma_finalize_kernel<true>, dim3(L * F), dim3(512), 0, ctx->stream, p, D, C, nt));
    else TACG_CUDA_TRY(ctx, tacg_launch_pdl(coact_mma_finalize_kernel<false>, dim3(L * F), dim3(512), 0, ctx->stream, p, D, C, nt));
    TACG_LAUNCH_CHECK(ctx);
    return TACG_OK;
}
