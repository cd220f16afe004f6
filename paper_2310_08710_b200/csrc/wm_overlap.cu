// a3 collision metric: pairwise oriented-box overlap by the separating-axis
// test, warp-tiled over the A x A matrix with symmetric-pair skipping: a warp takes a
// 32 x 32 tile (I, J) with I <= J, lane l holds agent j = 32 J + l in registers and walks the
// 32 agents i of block I (broadcast from shared memory).  One ballot gives word J of row i,
// and each lane accumulates word I of its own row j, so a tile fills both triangles.
// FP32-ALU bound (~40 flop per unordered pair), < 1 % of the step.
#include "wm_device.cuh"

struct OverlapParams {
  wm_row row;
  int A, W;               // W = ceil(A/32) words per row
  uint32_t* pair_bits;    // [B][A][W] or NULL
  uint8_t* flag; int64_t flag_stride_b;
};

__global__ void __launch_bounds__(1024) k_overlap(OverlapParams p) {
  extern __shared__ float sm[];
  const int A = p.A, nb = p.W, Ap = nb * 32;
  float* sx = sm;            float* sy = sx + Ap;
  float* sc = sy + Ap;       float* ss = sc + Ap;
  float* shl = ss + Ap;      float* shw = shl + Ap;
  float* srad = shw + Ap;                     // circumradius
  uint32_t* svalid = (uint32_t*)(srad + Ap);  // [nb] ballot words
  uint32_t* sany = svalid + nb;               // [Ap] any-overlap per agent
  const int b = blockIdx.y;
  const int64_t ro = (int64_t)b * p.row.stride_b;
  for (int a = threadIdx.x; a < Ap; a += blockDim.x) {
    const bool v = a < A && p.row.valid[ro + a] != 0;
    float x = 0.f, y = 0.f, c = 1.f, s = 0.f, hl = 0.f, hw = 0.f;
    if (v) {
      x = p.row.x[ro + a]; y = p.row.y[ro + a];
      sincosf(p.row.yaw[ro + a], &s, &c);
      hl = 0.5f * p.row.length[ro + a]; hw = 0.5f * p.row.width[ro + a];
    }
    sx[a] = x; sy[a] = y; sc[a] = c; ss[a] = s; shl[a] = hl; shw[a] = hw;
    srad[a] = sqrtf(fmaf(hl, hl, hw * hw));
    sany[a] = 0;
    const uint32_t w = __ballot_sync(0xffffffffu, v);
    if ((a & 31) == 0) svalid[a >> 5] = w;
  }
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  const int ntile = nb * (nb + 1) / 2;
  // gridDim.x > 1 (large A): the CTAs of a scenario split the tiles, nw consecutive ones each
  const int tile_lo = gridDim.x > 1 ? blockIdx.x * nw : 0, tile_hi = gridDim.x > 1 ? min(ntile, tile_lo + nw) : ntile;
  for (int tile = tile_lo + warp; tile < tile_hi; tile += nw) {
    // unrank (I <= J) from the linear upper-triangle index
    int I = 0, rem = tile;
    while (rem >= nb - I) { rem -= nb - I; ++I; }
    const int J = I + rem;
    const uint32_t vi = svalid[I], vj = svalid[J];
    uint32_t colword = 0, rowword = 0;
    if (vi != 0 && vj != 0) {
      const int j = J * 32 + lane;
      const float xj = sx[j], yj = sy[j], cj = sc[j], sj = ss[j], hlj = shl[j], hwj = shw[j], rj = srad[j];
      const bool jv = (vj >> lane) & 1u;
      for (int ii = 0; ii < 32; ++ii) {
        if (!((vi >> ii) & 1u)) continue;          // warp-uniform skip of invalid i
        const int i = I * 32 + ii;
        const float dx = xj - sx[i], dy = yj - sy[i];
        // off-diagonal tiles have i < j; a diagonal tile takes each unordered pair once, as (i < j):
        // the lower index is always in the i role, so overlap(i, j) == overlap(j, i) bit for bit
        // (the fused rollout kernel evaluates pairs in this order as well, P14)
        bool ov = jv && i < j && wm_circles_touch(dx, dy, rj + srad[i]);
        if (!__any_sync(0xffffffffu, ov)) continue;                   // far apart: row word stays 0
        ov = ov && wm_sat_overlap(dx, dy, sc[i], ss[i], shl[i], shw[i], cj, sj, hlj, hwj);
        const uint32_t w = __ballot_sync(0xffffffffu, ov);
        if (lane == ii) rowword = w;               // word J of row i
        colword |= (ov ? 1u : 0u) << ii;           // word I of row j
      }
    }
    const int i_mine = I * 32 + lane, j_mine = J * 32 + lane;
    if (I == J) { rowword |= colword; colword = 0; }         // the diagonal word holds both triangles
    if (p.pair_bits) {
      if (i_mine < A) p.pair_bits[((int64_t)b * A + i_mine) * nb + J] = rowword;
      if (I != J && j_mine < A) p.pair_bits[((int64_t)b * A + j_mine) * nb + I] = colword;
    }
    if (rowword) atomicOr(&sany[i_mine], 1u);
    if (colword) atomicOr(&sany[j_mine], 1u);
  }
  __syncthreads();
  if (gridDim.x == 1) {
    for (int a = threadIdx.x; a < A; a += blockDim.x) p.flag[(int64_t)b * p.flag_stride_b + a] = (uint8_t)(sany[a] != 0);
  } else {                                       // flags were zeroed by the launcher: OR this CTA's part in, byte a of a 4-byte word
    uint8_t* row = p.flag + (int64_t)b * p.flag_stride_b;
    for (int a = threadIdx.x; a < A; a += blockDim.x)
      if (sany[a] != 0) atomicOr((unsigned int*)(row + (a & ~3)), 1u << (8 * (a & 3)));
  }
}

cudaError_t wm_launch_overlap(wm_handle* h, const wm_traj& sim, int t, uint32_t* pair_bits,
                              uint8_t* flag, int64_t flag_stride_b, cudaStream_t s) {
  OverlapParams p;
  p.row = wm_make_row(sim, t);
  p.A = sim.A; p.W = (sim.A + 31) / 32;
  p.pair_bits = pair_bits; p.flag = flag; p.flag_stride_b = flag_stride_b;
  const int Ap = p.W * 32;
  const size_t smem = (size_t)Ap * 8 * 4 + (size_t)p.W * 4;
  // one warp per 32 x 32 tile of the upper triangle, up to 32 warps per scenario (A = 512: 136 tiles)
  const int ntile = p.W * (p.W + 1) / 2;
  const int nt = ntile >= 32 ? 1024 : (ntile > 8 ? 512 : 256);
  // More than 32 tiles (A > 224) and few scenarios: several CTAs per scenario, flags combined by atomic OR
  // on 4-byte words of the (zeroed) flag rows - needs 4-byte aligned rows.
  int split = 1;
  if (ntile > 32 && sim.B < 4 * h->num_sms && ((uintptr_t)flag & 3u) == 0 && flag_stride_b % 4 == 0 && sim.A % 4 == 0) split = (ntile + 31) / 32;
  if (split > 1) {
    cudaError_t e = flag_stride_b == sim.A ? cudaMemsetAsync(flag, 0, (size_t)sim.B * sim.A, s)
                                           : cudaMemset2DAsync(flag, (size_t)flag_stride_b, 0, (size_t)sim.A, (size_t)sim.B, s);
    if (e != cudaSuccess) return e;
  }
  k_overlap<<<dim3(split, sim.B), nt, smem, s>>>(p);
  h->launches++;
  return cudaGetLastError();
}
