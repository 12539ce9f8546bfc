// potential_tc.cu -- K1, the structure-factor potential, as a tensor-core contraction (tcgen05 / TMEM, sm_100a).
//
//   V_n[h,k] = sum_s f_s(q^2) sum_{j in (n,s)} exp(-2 pi i h u_j) exp(-2 pi i k v_j)                   (O2)
// With ex_j[h] = a + i b and ey_j[k] = c + i d the four real sums  ac, ad, bc, bd  over the atoms of a slice give all four
// quadrants of V (potential.cu, quadrant form).  Stacking A = [a ; b] (128 rows: 64 values of h, real and imaginary part)
// and B = [c ; d] (128 rows: 64 values of k), those sums are ONE real matrix product per species,
//       D[128 x 128] = A[128 x K] . B[128 x K]^T,      K = atoms of that species in the slice,
// the only dense contraction on the TACAW path (north_star (1)).  It runs here on the 5th-generation
// tensor cores: tcgen05.mma kind::tf32 issued by one thread, operands in shared memory in the canonical K-major
// no-swizzle layout, accumulators in tensor memory (one 128-column block per species), read back with tcgen05.ld.
// Accuracy: a tf32 operand keeps 11 significant bits, far short of the 2e-6 the transmission needs, so every operand is
// split x = hi + lo (hi = x with the low 13 mantissa bits cleared, lo = x - hi exactly) and each k-step issues the three
// products hi.hi + hi.lo + lo.hi ("3xTF32"; the dropped lo.lo term is 2^-22 relative), accumulated in fp32 in TMEM.
// Operands are generated in the kernel from the fixed-point fractional coordinates (exact two-level phases, as in the
// fp32-pipe kernel), so nothing but the sorted coordinates is read and V is written once.
#include "ctx.h"

namespace tacaw {

namespace {

constexpr int TC_TILE = 64;        // values of h (and of k) per CTA tile: 128 operand rows with real and imaginary parts
constexpr int TC_KB = 16;          // atoms per pipeline stage (two k-steps of 8)
constexpr int TC_THREADS = 128;
constexpr int TC_MAX_SPECIES = 4;  // 4 x 128 accumulator columns = all 512 TMEM columns
constexpr int TC_OPER_BYTES = 128 * TC_KB * 4;     // one operand block: 128 rows x 16 atoms of tf32 = 8 KB
constexpr int TC_STAGE_BYTES = 4 * TC_OPER_BYTES;  // A_hi, A_lo, B_hi, B_lo

__device__ __forceinline__ unsigned s32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// Shared-memory matrix descriptor, K-major, no swizzle: 8-row x 16-byte core matrices, the rows of a k-chunk contiguous
// (16 B apart), 8-row groups 128 B apart (stride byte offset), the two k-chunks of a k-step one operand column apart
// (leading byte offset = 128 rows x 16 B).  Bit layout: start address [0,14), LBO [16,30), SBO [32,46) (all >> 4),
// descriptor version 1 for sm_100 at [46,48), layout type 0 (no swizzle) at [61,64).
__device__ __forceinline__ unsigned long long smem_desc(unsigned addr) {
    const unsigned long long lbo = (128 * 16) >> 4, sbo = (8 * 16) >> 4;
    return (unsigned long long)((addr & 0x3FFFF) >> 4) | (lbo << 16) | (sbo << 32) | (1ull << 46);
}
// Instruction descriptor, kind::tf32: D format f32 (1 at [4,6)), A and B format tf32 (2 at [7,10) and [10,13)), both K-major,
// N >> 3 at [17,23), M >> 4 at [24,29).
constexpr unsigned TC_IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((128u >> 3) << 17) | ((128u >> 4) << 24);

__device__ __forceinline__ void mma_tf32(unsigned d_tmem, unsigned long long da, unsigned long long db, unsigned accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(da), "l"(db), "r"(TC_IDESC), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void mma_commit(unsigned long long* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(s32(bar)) : "memory");
}
__device__ __forceinline__ void bar_init(unsigned long long* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(s32(bar)), "r"(count) : "memory");
}
// bounded wait: a miscounted barrier traps after ~2 s instead of hanging the GPU
__device__ __forceinline__ void bar_wait(unsigned long long* bar, unsigned parity) {
    const unsigned a = s32(bar);
    const long long t0 = clock64();
    for (;;) {
        unsigned ok;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
        if (ok) return;
        if (clock64() - t0 > 4000000000LL) asm volatile("trap;");
    }
}

__device__ __forceinline__ float2 phase_fx(uint32_t u, int h) {      // exp(-2 pi i h u/2^32), exact argument reduction
    const int32_t p = (int32_t)((uint32_t)h * u);
    float s, c;
    sincospif((float)p * 4.656612873077393e-10f, &s, &c);
    return make_float2(c, -s);
}
__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }

constexpr int TC_ATOMS_SMEM = 2048; // sorted coordinates of a species staged per pass (16 KB)

struct TcSmem {
    // rows padded to 17 entries (136 B): the 8 rows a quarter-warp reads start in different banks
    float2 coarse[2][2][8][TC_KB + 1]; // [stage][axis][tile row / 8][atom]: exp(-2 pi i (x0 + 8 c) u)
    float2 fine[2][2][8][TC_KB + 1];   //                 [tile row % 8]     exp(-2 pi i f u)
    uint32_t ux[TC_ATOMS_SMEM], uy[TC_ATOMS_SMEM];   // fixed-point coordinates of the species being accumulated
    float gk[TC_MAX_SPECIES][4][TC_TILE];   // exp(-b_sg k^2/ly^2) for the tile's k
    unsigned long long bar_stage[2];   // MMAs that read a stage have completed
    unsigned long long bar_done;       // all MMAs of the tile have completed
    unsigned tmem_base;
};

}  // namespace

// One CTA = one (64 h) x (64 k) tile of the quadrant h, k >= 0 of one slice.  All 128 threads generate operands; thread 0
// issues the MMAs of a stage while the CTA generates the next one (two stages; tcgen05.commit on the stage's mbarrier
// releases its buffers).  Epilogue: TMEM -> registers, species sum with f_s, the two halves (real-part rows and
// imaginary-part rows of A) meet through shared memory, four quadrant stores per point.
__global__ void __launch_bounds__(TC_THREADS) k_potential_tc(const uint32_t* __restrict__ sx, const uint32_t* __restrict__ sy,
                                                              const int* __restrict__ offsets, int nspecies, const AbTable ab,
                                                              const int* __restrict__ kmax_pot, int hmax, int nx, int ny,
                                                              float inv_lx, float inv_ly, float2* __restrict__ V) {
    extern __shared__ __align__(1024) unsigned char dyn[];
    TcSmem& sm = *reinterpret_cast<TcSmem*>(dyn + 2 * TC_STAGE_BYTES);
    const int n = blockIdx.z;
    const int h0 = blockIdx.x * TC_TILE, k0 = blockIdx.y * TC_TILE;
    if (h0 > hmax || kmax_pot[h0] < k0) return;        // tile entirely outside the mask (uniform for the CTA)
    const int lt = threadIdx.x, warp = lt >> 5, lane = lt & 31;
    const int ncols = nspecies <= 1 ? 128 : (nspecies == 2 ? 256 : 512);

    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(s32(&sm.tmem_base)), "r"(ncols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (lt == 32) {
        bar_init(&sm.bar_stage[0], 1);
        bar_init(&sm.bar_stage[1], 1);
        bar_init(&sm.bar_done, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = lt; i < nspecies * 4 * TC_TILE; i += TC_THREADS) {
        const int j = i % TC_TILE, g = (i / TC_TILE) % 4, s = i / (4 * TC_TILE);
        const float qy = (float)(k0 + j) * inv_ly;
        sm.gk[s][g][j] = expf(-ab.b[s][g] * qy * qy);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem = sm.tmem_base;

    // ---- main loop: k-blocks of TC_KB atoms, species by species ----
    const int row = lt & 63;                 // tile row (value of h for A, of k for B) this thread generates
    const int half = lt >> 6;                // which 8 of the stage's 16 atoms
    int it = 0;                              // k-blocks issued so far (stage = it & 1)
    unsigned ph[2] = {0, 0};                 // parity of the next completion to wait for, per stage
    unsigned used = 0;                       // bit s: species s has atoms in this slice
    for (int s = 0; s < nspecies; ++s) {
        const int a0 = offsets[n * nspecies + s], a1 = offsets[n * nspecies + s + 1];
        if (a0 == a1) continue;
        used |= 1u << s;
        const unsigned d_tmem = tmem + 128u * s;
        for (int base = a0; base < a1; base += TC_KB, ++it) {
            const int st = it & 1;
            const int cnt = min(TC_KB, a1 - base);
            // coordinates: one coalesced pass per TC_ATOMS_SMEM atoms instead of a dependent global load per k-block
            const int rel = (base - a0) % TC_ATOMS_SMEM;
            if (rel == 0) {
                __syncthreads();                 // the previous pass's coordinates are no longer being read
                const int nload = min(TC_ATOMS_SMEM, a1 - base);
                for (int i = lt; i < nload; i += TC_THREADS) { sm.ux[i] = sx[base + i]; sm.uy[i] = sy[base + i]; }
                __syncthreads();
            }
            if (it >= 2) {                   // the MMAs that read this stage two k-blocks ago must be done
                bar_wait(&sm.bar_stage[st], ph[st]);
                ph[st] ^= 1;
            }
            // phase tables of the stage: 16 atoms x 2 axes x (8 coarse + 8 fine) = 512 entries
            for (int i = lt; i < TC_KB * 32; i += TC_THREADS) {
                const int at = i % TC_KB, e = i / TC_KB;        // e: axis*16 + table entry
                const int axis = e >> 4, j = e & 15;
                float2 v = make_float2(0.f, 0.f);               // atoms past the end of the species contribute nothing
                if (at < cnt) {
                    const uint32_t u = axis ? sm.uy[rel + at] : sm.ux[rel + at];
                    v = (j < 8) ? phase_fx(u, (axis ? k0 : h0) + 8 * j) : phase_fx(u, j - 8);
                }
                if (j < 8) sm.coarse[st][axis][j][at] = v; else sm.fine[st][axis][j - 8][at] = (at < cnt) ? v : make_float2(0.f, 0.f);
            }
            __syncthreads();
            // operand blocks of the stage: element (row r, atom a) of a block sits at (a/4)*2048 + r*16 + (a%4)*4 bytes
            unsigned char* stage = dyn + st * TC_STAGE_BYTES;
#pragma unroll
            for (int axis = 0; axis < 2; ++axis) {
                float* hi = reinterpret_cast<float*>(stage + (axis ? 2 : 0) * TC_OPER_BYTES);
                float* lo = reinterpret_cast<float*>(stage + (axis ? 3 : 1) * TC_OPER_BYTES);
#pragma unroll
                for (int ch = 0; ch < 2; ++ch) {
                    const int kc = half * 2 + ch;                // 16-byte k-chunk of the stage (4 atoms)
                    float re[4], im[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int at = kc * 4 + q;
                        const float2 cph = sm.coarse[st][axis][row >> 3][at], fph = sm.fine[st][axis][row & 7][at];
                        re[q] = cph.x * fph.x - cph.y * fph.y;
                        im[q] = cph.x * fph.y + cph.y * fph.x;
                    }
                    float4 rh, rl, ih, il;
                    rh.x = tf32_hi(re[0]); rh.y = tf32_hi(re[1]); rh.z = tf32_hi(re[2]); rh.w = tf32_hi(re[3]);
                    rl.x = re[0] - rh.x;   rl.y = re[1] - rh.y;   rl.z = re[2] - rh.z;   rl.w = re[3] - rh.w;
                    ih.x = tf32_hi(im[0]); ih.y = tf32_hi(im[1]); ih.z = tf32_hi(im[2]); ih.w = tf32_hi(im[3]);
                    il.x = im[0] - ih.x;   il.y = im[1] - ih.y;   il.z = im[2] - ih.z;   il.w = im[3] - ih.w;
                    const int o_re = (kc * 2048 + row * 16) >> 2, o_im = (kc * 2048 + (64 + row) * 16) >> 2;
                    *reinterpret_cast<float4*>(hi + o_re) = rh;
                    *reinterpret_cast<float4*>(lo + o_re) = rl;
                    *reinterpret_cast<float4*>(hi + o_im) = ih;
                    *reinterpret_cast<float4*>(lo + o_im) = il;
                }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic-proxy writes -> visible to the MMA
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncthreads();
            if (lt == 0) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const unsigned sa = s32(stage);
#pragma unroll
                for (int ks = 0; ks < TC_KB / 8; ++ks) {
                    // a k-step of 8 atoms = two 16-byte chunks = 4096 bytes further into each operand block
                    const unsigned long long a_hi = smem_desc(sa + 0 * TC_OPER_BYTES + ks * 4096);
                    const unsigned long long a_lo = smem_desc(sa + 1 * TC_OPER_BYTES + ks * 4096);
                    const unsigned long long b_hi = smem_desc(sa + 2 * TC_OPER_BYTES + ks * 4096);
                    const unsigned long long b_lo = smem_desc(sa + 3 * TC_OPER_BYTES + ks * 4096);
                    mma_tf32(d_tmem, a_hi, b_hi, (base > a0 || ks > 0) ? 1u : 0u);
                    mma_tf32(d_tmem, a_hi, b_lo, 1u);
                    mma_tf32(d_tmem, a_lo, b_hi, 1u);
                }
                mma_commit(&sm.bar_stage[st]);       // arrives when these MMAs (and all earlier ones) have completed
            }
        }
    }
    if (lt == 0) mma_commit(&sm.bar_done);
    bar_wait(&sm.bar_done, 0);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

    // ---- epilogue ----
    // TMEM lane = operand row of A: lanes 0..63 hold (ac | ad) for h = h0 + lane (columns 0..63 | 64..127 of a species block),
    // lanes 64..127 hold (bc | bd).  Warp w reads lanes 32 w .. 32 w + 31.
    const int hrow = lt & 63;
    const int h = h0 + hrow;
    const bool low = lt < 64;                 // real-part rows
    float gh[TC_MAX_SPECIES][4];
#pragma unroll
    for (int s = 0; s < TC_MAX_SPECIES; ++s)
#pragma unroll
        for (int g = 0; g < 4; ++g) {
            const float qx = (float)h * inv_lx;
            gh[s][g] = (s < nspecies) ? ab.a[s][g] * expf(-ab.b[s][g] * qx * qx) : 0.f;
        }
    float2* xch = reinterpret_cast<float2*>(dyn);        // [16 columns][64 rows] (bc, bd) of the imaginary-part rows; stage buffers are idle
    float2* Vn = V + (size_t)n * nx * ny;
    const int kmh = (h <= hmax) ? kmax_pot[h] : -1;
    for (int jc = 0; jc < TC_TILE; jc += 16) {
        float p1[16], p2[16];                 // species-summed (ac, ad) or (bc, bd) for columns jc .. jc + 15
#pragma unroll
        for (int j = 0; j < 16; ++j) p1[j] = p2[j] = 0.f;
#pragma unroll
        for (int s = 0; s < TC_MAX_SPECIES; ++s) {
            if (s < nspecies && ((used >> s) & 1u)) {
                unsigned r1[16], r2[16];
                const unsigned ta = tmem + ((unsigned)(warp * 32) << 16) + 128u * s + jc;
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                             : "=r"(r1[0]), "=r"(r1[1]), "=r"(r1[2]), "=r"(r1[3]), "=r"(r1[4]), "=r"(r1[5]), "=r"(r1[6]), "=r"(r1[7]),
                               "=r"(r1[8]), "=r"(r1[9]), "=r"(r1[10]), "=r"(r1[11]), "=r"(r1[12]), "=r"(r1[13]), "=r"(r1[14]), "=r"(r1[15])
                             : "r"(ta));
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                             : "=r"(r2[0]), "=r"(r2[1]), "=r"(r2[2]), "=r"(r2[3]), "=r"(r2[4]), "=r"(r2[5]), "=r"(r2[6]), "=r"(r2[7]),
                               "=r"(r2[8]), "=r"(r2[9]), "=r"(r2[10]), "=r"(r2[11]), "=r"(r2[12]), "=r"(r2[13]), "=r"(r2[14]), "=r"(r2[15])
                             : "r"(ta + 64u));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    float f = 0.f;
#pragma unroll
                    for (int g = 0; g < 4; ++g) f = fmaf(gh[s][g], sm.gk[s][g][jc + j], f);
                    p1[j] = fmaf(f, __uint_as_float(r1[j]), p1[j]);
                    p2[j] = fmaf(f, __uint_as_float(r2[j]), p2[j]);
                }
            }
        }
        __syncthreads();                      // previous chunk's exchange consumed
        if (!low) {
#pragma unroll
            for (int j = 0; j < 16; ++j) xch[j * 64 + hrow] = make_float2(p1[j], p2[j]);
        }
        __syncthreads();
        if (low && kmh >= 0) {
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const int k = k0 + jc + j;
                if (k > kmh) continue;
                const float2 q = xch[j * 64 + hrow];
                const float ac = p1[j], ad = p2[j], bc = q.x, bd = q.y;
                const int ixm = (nx - h) % nx, iym = (ny - k) % ny;
                Vn[(size_t)k * nx + h] = make_float2(ac - bd, ad + bc);
                if (k > 0) Vn[(size_t)iym * nx + h] = make_float2(ac + bd, bc - ad);
                if (h > 0) Vn[(size_t)iym * nx + ixm] = make_float2(ac - bd, -(ad + bc));
                if (h > 0 && k > 0) Vn[(size_t)k * nx + ixm] = make_float2(ac + bd, ad - bc);
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(ncols) : "memory");
    }
}

size_t potential_tc_smem() { return 2 * (size_t)TC_STAGE_BYTES + sizeof(TcSmem) + 1024; }
int potential_tc_max_species() { return TC_MAX_SPECIES; }

int launch_potential_tc(tacaw_ctx* ctx, const uint32_t* sx, const uint32_t* sy, const int* offsets, int nspecies, const AbTable& ab,
                        int nslices_total, float2* d_V, cudaStream_t st) {
    const int nx = ctx->grid.nx, ny = ctx->grid.ny;
    const size_t smem = potential_tc_smem();
    const void* key = (const void*)k_potential_tc;
    if (ctx->kernel_occ.find(key) == ctx->kernel_occ.end()) {
        TACAW_CUDA(ctx, cudaFuncSetAttribute(k_potential_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ctx->kernel_occ.emplace(key, 1);
    }
    const int hmax = ctx->hmax_pot;
    for (int z0 = 0; z0 < nslices_total; z0 += 65535) {
        const int nz = nslices_total - z0 < 65535 ? nslices_total - z0 : 65535;
        dim3 grid((hmax + TC_TILE) / TC_TILE, (ctx->kmaxmax_pot + TC_TILE) / TC_TILE, nz);
        k_potential_tc<<<grid, TC_THREADS, smem, st>>>(sx, sy, offsets + (size_t)z0 * nspecies, nspecies, ab, ctx->d_kmax_pot, hmax, nx, ny,
                                                       (float)(1.0 / ctx->grid.lx_A), (float)(1.0 / ctx->grid.ly_A),
                                                       d_V + (size_t)z0 * nx * ny);
        ctx->launches++;
    }
    TACAW_CUDA(ctx, cudaGetLastError());
    return TACAW_OK;
}

}  // namespace tacaw
