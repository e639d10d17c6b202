// rbq_diag.cu -- diagnostics that are not a stage of the path: the row-gather experiment of SURVEY.md section 7, hard
// part 5 ("random 256-B row gathers at >= 70 % of HBM": TMA tile::gather4 against cp.async staging), kept in the library so
// that its numbers (bench.py leg `gather4_experiment`, profiles/r02_ncu.md) come from committed code.
//
// rbq_diag_gather streams the rows `rows[0 .. n)` of two bf16 matrices K and V ([n_rows_total][D], D = 128: 256-byte rows,
// the layout of one (sequence, KV head) slab of the cache) through shared memory exactly as attn_gather_kernel does -- one
// persistent CTA per SM, 8 warps, a private 3-stage ring of 16-row K + V tiles per warp (192 KB in flight per SM) -- and
// folds what landed into a 64-bit checksum instead of contracting it.
//   mode 0: 16-byte cp.async (LDGSTS) per lane, 32 per lane and tile, as in the product kernel;
//   mode 1: cp.async.bulk.tensor.2d ... tile::gather4 (UTMALDG.2D.GATHER4): 4 rows by index per instruction, issued by
//           one lane, completion on an mbarrier per stage;
//   modes 2 / 3: the same two on ONE matrix of interleaved K | V rows ([n_rows_total][256], 512-byte rows; V is ignored):
//           half as many instructions per byte for the TMA form (4 x 512 B each).
#include <cuda.h>

#include "rbq_common.cuh"

namespace {

constexpr int DG_WARPS = 8, DG_THREADS = DG_WARPS * 32, DG_STAGES = 3, DG_TILE = 16, DG_D = 128;
constexpr int DG_ROW_BYTES = DG_D * 2, DG_TILE_BYTES = DG_TILE * DG_ROW_BYTES, DG_STAGE_BYTES = 2 * DG_TILE_BYTES;
constexpr int DG_SMEM = DG_WARPS * DG_STAGES * DG_STAGE_BYTES;   // 192 KB

__device__ __forceinline__ unsigned long long fold16(uint32_t addr) {
  uint32_t a, b, c, d;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "r"(addr));
  return (unsigned long long)a + b + c + d;
}

#define RBQ_DG_GATHER4(dst, map, bar, r0_, r1_, r2_, r3_)                                                                   \
  asm volatile(                                                                                                             \
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile::gather4.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];" \
      ::"r"(dst), "l"(map), "r"(bar), "r"(0), "r"(r0_), "r"(r1_), "r"(r2_), "r"(r3_) : "memory")

template <int MODE>
__global__ void __launch_bounds__(DG_THREADS, 1)
diag_gather_kernel(const __nv_bfloat16* __restrict__ K, const __nv_bfloat16* __restrict__ V,
                   const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                   const int32_t* __restrict__ rows, long long n, unsigned long long* __restrict__ checksum) {
  extern __shared__ __align__(1024) unsigned char dg_smem[];
  __shared__ __align__(8) unsigned long long s_bar[DG_WARPS][DG_STAGES];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long r0 = n * blockIdx.x / gridDim.x, r1 = n * (blockIdx.x + 1) / gridDim.x;
  const int cnt = (int)(r1 - r0);
  const int ntiles = (cnt + DG_TILE - 1) / DG_TILE;
  const int my_tiles = ntiles > warp ? (ntiles - warp + DG_WARPS - 1) / DG_WARPS : 0;
  const uint32_t my_base = rbq_smem_u32(dg_smem + (size_t)warp * DG_STAGES * DG_STAGE_BYTES);
  constexpr bool TMA = (MODE & 1) != 0, IL = MODE >= 2;           // IL: interleaved K | V rows of 512 bytes
  if (TMA) {
    if (lane == 0)
      for (int s = 0; s < DG_STAGES; ++s) rbq_mbar_init(rbq_smem_u32(&s_bar[warp][s]), 1);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
  }
  auto entry = [&](int i) -> int {                               // row of lane (< 16) of tile i of this warp, -1 = padding
    const long long r = r0 + (long long)(warp + i * DG_WARPS) * DG_TILE + lane;
    return (lane < DG_TILE && r < r1) ? rows[r] : -1;
  };
  auto issue = [&](int i, int ent) {
    const uint32_t sbase = my_base + (uint32_t)((i % DG_STAGES) * DG_STAGE_BYTES);
    if (!TMA) {
      if (!IL) {
#pragma unroll
        for (int k = 0; k < DG_TILE / 2; ++k) {                  // 32 lanes cover 2 rows of 16 chunks per step
          const int row = 2 * k + (lane >> 4), ch = lane & 15;
          const int re = __shfl_sync(0xffffffffu, ent, row);
          const long long off = (long long)max(re, 0) * DG_D + ch * 8;
          const uint32_t d = sbase + (uint32_t)(row * DG_ROW_BYTES + (ch << 4));
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(K + off) : "memory");
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d + DG_TILE_BYTES), "l"(V + off) : "memory");
        }
      } else {
#pragma unroll
        for (int row = 0; row < DG_TILE; ++row) {                // 32 lanes cover one 512-byte row per step
          const int re = __shfl_sync(0xffffffffu, ent, row);
          const long long off = (long long)max(re, 0) * (2 * DG_D) + lane * 8;
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sbase + (uint32_t)(row * 2 * DG_ROW_BYTES + (lane << 4))), "l"(K + off) : "memory");
        }
      }
      asm volatile("cp.async.commit_group;" ::: "memory");
    } else {
      int e[DG_TILE];
#pragma unroll
      for (int k = 0; k < DG_TILE; ++k) e[k] = max(__shfl_sync(0xffffffffu, ent, k), 0);
      if (lane == 0) {
        const uint32_t bar = rbq_smem_u32(&s_bar[warp][i % DG_STAGES]);
        rbq_mbar_expect_tx(bar, (uint32_t)DG_STAGE_BYTES);
#pragma unroll
        for (int k = 0; k < DG_TILE / 4; ++k) {
          if (!IL) {
            RBQ_DG_GATHER4(sbase + (uint32_t)(4 * k * DG_ROW_BYTES), &tmK, bar, e[4 * k], e[4 * k + 1], e[4 * k + 2], e[4 * k + 3]);
            RBQ_DG_GATHER4(sbase + (uint32_t)(DG_TILE_BYTES + 4 * k * DG_ROW_BYTES), &tmV, bar, e[4 * k], e[4 * k + 1], e[4 * k + 2], e[4 * k + 3]);
          } else {
            RBQ_DG_GATHER4(sbase + (uint32_t)(4 * k * 2 * DG_ROW_BYTES), &tmK, bar, e[4 * k], e[4 * k + 1], e[4 * k + 2], e[4 * k + 3]);
          }
        }
      }
    }
  };
  unsigned long long acc = 0;
  int ent_next[DG_STAGES];
#pragma unroll
  for (int s = 0; s < DG_STAGES; ++s) ent_next[s] = s < my_tiles ? entry(s) : -1;
#pragma unroll
  for (int s = 0; s < DG_STAGES - 1; ++s) {
    if (s < my_tiles) issue(s, ent_next[s]);
    else if (!TMA) asm volatile("cp.async.commit_group;" ::: "memory");
  }
  for (int i = 0; i < my_tiles; ++i) {
    const int nx = i + DG_STAGES - 1;
    const int ent_cur = ent_next[0];
#pragma unroll
    for (int s = 0; s + 1 < DG_STAGES; ++s) ent_next[s] = ent_next[s + 1];
    if (nx < my_tiles) issue(nx, ent_next[DG_STAGES - 2]);
    else if (!TMA) asm volatile("cp.async.commit_group;" ::: "memory");
    ent_next[DG_STAGES - 1] = (nx + 1 < my_tiles) ? entry(nx + 1) : -1;
    const uint32_t sbase = my_base + (uint32_t)((i % DG_STAGES) * DG_STAGE_BYTES);
    if (!TMA) {
      asm volatile("cp.async.wait_group %0;" ::"n"(DG_STAGES - 1) : "memory");
      __syncwarp();
    } else {
      rbq_mbar_wait(rbq_smem_u32(&s_bar[warp][i % DG_STAGES]), (uint32_t)((i / DG_STAGES) & 1));
    }
    // fold the valid rows: lane -> (row = lane >> 1, half = lane & 1): 16 chunks of 16 bytes (8 of K and 8 of V, or 16 of
    // the interleaved row)
    const int row = lane >> 1;
    const int re = __shfl_sync(0xffffffffu, ent_cur, row);
    if (re >= 0) {
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        if (!IL) {
          const uint32_t a = sbase + (uint32_t)(row * DG_ROW_BYTES + (((lane & 1) * 8 + c) << 4));
          acc += fold16(a) + fold16(a + DG_TILE_BYTES);
        } else {
          const uint32_t a = sbase + (uint32_t)(row * 2 * DG_ROW_BYTES + (((lane & 1) * 16 + c) << 4));
          acc += fold16(a) + fold16(a + 128);
        }
      }
    }
    __syncwarp();                                              // tile consumed before its stage is refilled
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0 && acc) atomicAdd(checksum, acc);
}

typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                              const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                              CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 2-D map over [n_rows_total][width] bf16; tile::gather4 wants a box of ONE row, the instruction names four of them
int make_map(rbq_ctx* ctx, CUtensorMap* tm, const void* base, long long n_rows_total, int width) {
  void* f = nullptr;
  cudaDriverEntryPointQueryResult qres;
  RBQ_CUDA_OK(ctx, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qres));
  if (!f || qres != cudaDriverEntryPointSuccess) RBQ_FAIL(ctx, RBQ_ERR_UNSUPPORTED, "cuTensorMapEncodeTiled not available");
  const cuuint64_t gdim[2] = {(cuuint64_t)width, (cuuint64_t)n_rows_total};
  const cuuint64_t gstr[1] = {(cuuint64_t)width * 2};
  const cuuint32_t box[2] = {(cuuint32_t)width, 1u};
  const cuuint32_t estr[2] = {1u, 1u};
  const CUresult r = ((encode_fn)f)(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gdim, gstr, box, estr,
                                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) RBQ_FAIL(ctx, RBQ_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
  return RBQ_OK;
}

}  // namespace

int rbq_diag_gather(rbq_ctx* ctx, const void* K, const void* V, long long n_rows_total, const int32_t* rows, long long n,
                    int mode, unsigned long long* checksum, void* stream) {
  if (!ctx) return RBQ_ERR_INVALID_ARG;
  if (!K || !rows || !checksum || n < 0 || n_rows_total <= 0 || mode < 0 || mode > 3 || (mode < 2 && !V))
    RBQ_FAIL(ctx, RBQ_ERR_INVALID_ARG, "rbq_diag_gather: bad argument");
  cudaStream_t s = (cudaStream_t)stream;
  CUtensorMap tmK, tmV;
  memset(&tmK, 0, sizeof(tmK));
  memset(&tmV, 0, sizeof(tmV));
  if (mode & 1) {
    int rc = make_map(ctx, &tmK, K, n_rows_total, mode >= 2 ? 2 * DG_D : DG_D);
    if (rc != RBQ_OK) return rc;
    if (mode < 2) {
      rc = make_map(ctx, &tmV, V, n_rows_total, DG_D);
      if (rc != RBQ_OK) return rc;
    }
  }
#define RBQ_DIAG_LAUNCH(M)                                                                                         \
  do {                                                                                                             \
    RBQ_SET_SMEM_ATTR(ctx, RBQ_ATTR_MISC + 4 + M, diag_gather_kernel<M>, DG_SMEM);                                 \
    diag_gather_kernel<M><<<ctx->sm_count, DG_THREADS, DG_SMEM, s>>>((const __nv_bfloat16*)K, (const __nv_bfloat16*)V, tmK, tmV, rows, n, checksum); \
  } while (0)
  switch (mode) {
    case 0: RBQ_DIAG_LAUNCH(0); break;
    case 1: RBQ_DIAG_LAUNCH(1); break;
    case 2: RBQ_DIAG_LAUNCH(2); break;
    default: RBQ_DIAG_LAUNCH(3); break;
  }
#undef RBQ_DIAG_LAUNCH
  RBQ_LAUNCH_OK(ctx);
  return RBQ_OK;
}
