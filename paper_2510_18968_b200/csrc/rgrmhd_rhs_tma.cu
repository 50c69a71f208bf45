// rgrmhd_rhs_tma.cu -- the production flux-divergence kernel (a2, a3, divergence of a4, divergence part
// of a5) for sm_100a: reconstruct + HLLE + flux divergence + update of the stage target in ONE launch,
// with every reconstruction stencil staged in shared memory by the TMA engine.
//
// Decomposition: a CTA owns a TX x TY (x, y) tile of z-pencils and marches CZ planes along z; one
// compute thread = one cell of the current plane.  Per plane and direction K (x, y, z), for each of the
// 15 reconstructed variables, ONE bulk tensor copy (cp.async.bulk.tensor.4d, box = the tile plus its
// 3-cell halo along K only: (TX+6) x TY, (TX+2) x (TY+6) or (TX+2) x TY x 5 planes) lands in a ring of NS
// shared-memory stages.  A producer warp runs the ring ahead of the compute warps (full / empty
// mbarriers per stage), so no compute warp ever waits on a global load for a stencil:
//   a2  every compute thread reconstructs ITS OWN CELL along K from the staged box: the smoothness
//       indicators are computed once and give the value at the cell's lower face (a thread-private
//       shared-memory slot: the right state of that face) and at its upper face (shared memory: the left
//       state of the neighbour's face; along z it is carried to the next plane in a thread-private slot).  The 2 x 16 halo cells
//       of the tile are reconstructed by one warp per variable (round robin), from the same box.
//   a3  every compute thread solves the HLLE problem at its cell's lower face (x, y) / upper face (z);
//       the TX + TY faces on the tile's upper x / y edge are solved by a helper warp, concurrently.
//       Fluxes are exchanged through a second shared-memory buffer, so a phase needs two barriers.
//   a5  the increment dt dU or dt/2 dU is written once per cell (G.dU); the next recovery kernel adds it.
// The face metric (two cells x 8 fields) is prefetched into registers before the reconstruction loop.
// Warp roles: 8 compute warps, 1 producer warp (one lane issues the TMA copies), 1 edge-face warp, 2 halo
// warps: 12 warps = three per scheduler, the most that 168 registers per thread allow.
// The three directions run through ONE copy of the code (rgrmhd_flux_rot.cuh).
#include <cuda.h>

#include "rgrmhd_flux_rot.cuh"

namespace rg {

namespace {
constexpr int TX = 16, TY = 16, NT = TX * TY;
constexpr int NWC = NT / 32;                       // compute warps
constexpr int NHALO = 2;                            // halo-cell warps (variables dealt round robin)
constexpr int NTHREADS = NT + 64 + 32 * NHALO;     // + producer warp + edge-face warp + halo warps
constexpr int EXW = TX + 1, EXH = TY + 1, EXP = EXW * EXH;
constexpr int NS = 6;                              // ring stages
#ifndef RG_GROUP
#define RG_GROUP 2
#endif
constexpr int GR = RG_GROUP;                       // variables reconstructed per step (interleaved dependency chains)
// The TMA engine needs a 16-byte aligned box origin (an even x coordinate for doubles: an odd one traps with
// "illegal instruction"), and the ghost offset is 3: the y and z boxes therefore start one cell left of the tile
// and are TX + 2 wide.
constexpr int PY = TX + 2;                         // row pitch of the y and z boxes
constexpr int BOX_X = (TX + 6) * TY, BOX_Y = PY * (TY + 6), BOX_Z = PY * TY * 5;   // doubles per box
constexpr int STAGE_DBL = BOX_Z;
static_assert(BOX_X <= STAGE_DBL && BOX_Y <= STAGE_DBL, "stage must hold every box");
static_assert(TX == 16 && TY == 16, "halo / edge lane mapping assumes 16-lane rows and columns");

struct Smem {
  double ring[NS][STAGE_DBL];   // TMA destinations (128-byte aligned: STAGE_DBL * 8 is a multiple of 128)
  double ex[NVR][EXP];          // upper-face states of the tile's cells (+ lower halo): left states of the faces
  double fx[NCONS][EXP];        // face fluxes (slot = the cell whose lower face it is; column TX / row TY = edge)
  double exlo[NVR][16];         // lower-face states of the upper-halo cells (right states of the edge faces)
  double exhi[NVR][16];         // upper-face states of the last row/column (left states of the edge faces)
  double chi[NVR][NT];          // z carry: upper-face states of the plane below (thread-private slots)
  double los[NVR][NT];          // lower-face states of the own cell = right states of its face (thread-private slots)
  double du[NCONS][NT];         // flux divergence being accumulated for the current plane (thread-private)
  unsigned long long full[NS], empty[NS];
};

struct TmaMaps {
  CUtensorMap x, y, z;
};

// ---- mbarrier / TMA PTX ---------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* b, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned parity) {
  const unsigned a = smem_u32(b);
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "W_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra D_%=;\n"
      "bra W_%=;\n"
      "D_%=:\n"
      "}\n" ::"r"(a), "r"(parity) : "memory");
}
// one non-blocking probe: issue early, test the result later (the probe's ~90-cycle latency hides behind
// independent arithmetic)
__device__ __forceinline__ unsigned mbar_test(unsigned long long* b, unsigned parity) {
  unsigned ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n" : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
  return ok;
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_4d(const CUtensorMap* map, void* dst, unsigned long long* bar, int c0, int c1,
                                            int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}
// barrier among the compute warps and the edge-face warp (the producer warp never joins)
__device__ __forceinline__ void bar_work() { asm volatile("bar.sync 1, %0;" ::"n"(NT + 32 + 32 * NHALO) : "memory"); }
// barrier A ("face states visible") also has the halo warps, which write the halo states
__device__ __forceinline__ void bar_states() { asm volatile("bar.sync 2, %0;" ::"n"(NT + 32 + 32 * NHALO) : "memory"); }
__device__ __forceinline__ void prefetch_l2(const double* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
// pin a prefetched value in its register until here (keeps the consumer arithmetic below this point)
__device__ __forceinline__ void pin(double& x) { asm volatile("" : "+d"(x)); }

// rotated -> natural conserved index for K = 2 (rotated components 0,1,2 = z,x,y), known at compile time
__host__ __device__ constexpr int nat_z(int v) {
  return (v >= CSX && v <= CSZ) ? CSX + (v - CSX + 2) % 3
       : (v >= CEX && v <= CEZ) ? CEX + (v - CEX + 2) % 3
       : (v >= CBX && v <= CBZ) ? CBX + (v - CBX + 2) % 3 : v;
}

template <int RECON>
__device__ __forceinline__ void lds_stencil(const double* __restrict__ p, int s, double u[5]) {
  if (RECON == RECON_WENO5) { u[0] = p[-2 * s]; u[4] = p[2 * s]; } else { u[0] = 0.0; u[4] = 0.0; }
  u[1] = p[-s]; u[2] = p[0]; u[3] = p[s];
}
}  // namespace

template <int RECON, int CHARGE, int STAGE, int WAVE>
// 168 registers: 12 warps sit 3 + 3 + 3 + 3 on the four schedulers, each with a 16 K-register file
__global__ void __launch_bounds__(NTHREADS, 1)
k_flux_tma(const __grid_constant__ GridView G, const __grid_constant__ PencilTabs T,
           const __grid_constant__ TmaMaps M, double dt, int CZ) {
  constexpr int NV = (CHARGE == CHARGE_CELL_CURRENT) ? NVR : NVR - 1;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Smem& S = *reinterpret_cast<Smem*>(smem_raw);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int txn = min(TX, G.n[0] - i0), tyn = min(TY, G.n[1] - j0);   // valid extent of this tile
  const int k0 = blockIdx.z * CZ, k1 = min(k0 + CZ, G.n[2]);
  const long long sz = G.stride[2];
  if (tid == 0) {
#pragma unroll
    for (int q = 0; q < NS; ++q) { mbar_init(&S.full[q], 1); mbar_init(&S.empty[q], NWC + NHALO); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  // =================================================================================================
  // producer warp: one lane walks the (plane, direction, variable) sequence NS boxes ahead
  // =================================================================================================
  if (warp == NWC) {
    int pst = 0, pit = 0;                        // stage of the next box, uses of that stage so far
    for (int k = k0 - 2; k < k1; ++k) {
      if (lane == 0) {
        for (int K = (k < k0) ? 2 : 0; K < 3; ++K) {
          const CUtensorMap* map = (K == 0) ? &M.x : (K == 1) ? &M.y : &M.z;
          const unsigned bytes = 8u * (unsigned)((K == 0) ? BOX_X : (K == 1) ? BOX_Y : BOX_Z);
          // padded coordinates of the box origin (ghost offset 3): x box starts 3 cells left of the tile,
          // y box 3 rows below, z box at plane k-1 (stencil of cell k+1: planes k-1 .. k+3); y, z boxes start
          // one cell left of the tile (even x coordinate)
          const int px = i0 + ((K == 0) ? 0 : 2), py = j0 + ((K == 1) ? 0 : 3), pz = k + ((K == 2) ? 2 : 3);
          for (int vr = 0; vr < NV; ++vr) {
            // the refill of a released stage is on the consumers' critical path in the z phases: plain counters
            // and a spinning wait (measured 1 % faster than seq % NS and a suspended wait)
            const int st = pst, it = pit;
            if (++pst == NS) { pst = 0; ++pit; }
            if (it > 0) mbar_wait(&S.empty[st], (unsigned)(it - 1) & 1u);
            mbar_expect_tx(&S.full[st], bytes);
            tma_load_4d(map, S.ring[st], &S.full[st], px, py, pz, T.fld[K][vr]);
          }
        }
      } else {
        // The other lanes of this warp are idle: they pull the face-metric rows of the plane after the next one
        // into L2, so that the compute warps' loads of them two planes later are L2 hits instead of DRAM
        // accesses (no registers, no shared memory; paced by the issuing lane).
        const int kp = k + 2;
        if (kp >= k0 && kp < k1) {
          const int row = (lane - 1) >> 1, half = (lane - 1) & 1;    // 31 lanes: rows 0..14 twice + row 15 once
          for (int r = row; r < TY + 1; r += 16) {
            if (j0 + r - 1 >= G.n[1] + 1) continue;
            const long long cp = cell_index(G, i0 + half * 8, j0 + r - 1, kp);   // row r-1 (one halo row below the tile)
#pragma unroll
            for (int q = 0; q < 10; ++q) prefetch_l2(G.met[q] + cp);
          }
        }
      }
      __syncwarp();
    }
    return;
  }

  // =================================================================================================
  // edge-face warp: the TY faces on the tile's upper x edge and the TX faces on its upper y edge
  // =================================================================================================
  if (warp == NWC + 1) {
    const int r = lane & 15;
    for (int k = k0; k < k1; ++k) {
#pragma unroll 1
      for (int K = 0; K < 2; ++K) {
        const bool valid = lane < 16 && r < ((K == 0) ? tyn : txn);
        const long long cr = (K == 0) ? cell_index(G, i0 + txn, j0 + r, k) : cell_index(G, i0 + r, j0 + tyn, k);
        const long long cl = cr - G.stride[K];
        FaceRaw raw;
        if (valid) load_face_raw(T, K, cl, cr, raw);
        bar_states();                                                  // A: face states visible
        if (valid) {
          double PR[NVR], F[NCONS];
#pragma unroll
          for (int vr = 0; vr < NV; ++vr) PR[vr] = S.exlo[vr][r];
          FaceMet m;
          finish_face_met(raw, m);
          riemann_m<CHARGE, NV, WAVE>(G, m, cl, cr, &S.exhi[0][r], 16, PR, F);
          const int dst = (K == 0) ? r * EXW + txn : tyn * EXW + r;
#pragma unroll
          for (int v = 0; v < NCONS; ++v) S.fx[T.nat[K][v]][dst] = F[v];
        }
        bar_work();                                                    // C: fluxes visible
      }
    }
    return;
  }

  // =================================================================================================
  // halo warps: the 2 x 16 halo cells of the tile, one variable per warp and box (round robin); lanes 0-15 the
  // cells below the tile (their upper-face value), lanes 16-31 the cells above (their lower-face value)
  // =================================================================================================
  if (warp >= NWC + 2) {
    const int hw = warp - (NWC + 2);
    const int hr = lane & 15;
    const bool hup = lane >= 16;
    int st = 0;
    unsigned ph = 0;
    for (int k = k0 - 2; k < k1; ++k) {
#pragma unroll 1
      for (int K = (k < k0) ? 2 : 0; K < 3; ++K) {
        const int sst = (K == 0) ? 1 : PY;
        const int hal0 = (K == 0) ? hr * (TX + 6) + (hup ? txn + 3 : 2) : (hup ? tyn + 3 : 2) * PY + hr + 1;
        const bool hvalid = hr < ((K == 0) ? tyn : txn);
#pragma unroll 1
        for (int vr = 0; vr < NV; ++vr) {
          // every consumer warp observes and releases EVERY box (an mbarrier waiter that skips a phase cannot
          // tell it from the one two uses later); it reconstructs the halo cells only of its own variables
          {
            mbar_wait(&S.full[st], ph);
            const bool mine = K < 2 && vr % NHALO == hw;
            double u[1][5];
            if (mine) {
              lds_stencil<RECON>(&S.ring[st][hal0], sst, u[0]);
              asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            }
            // like the compute warps: the stage goes back to the producer as soon as the stencil is in registers
            __syncwarp();
            if (lane == 0) mbar_arrive(&S.empty[st]);
            if (mine) {
              // one face per halo cell: the upper face of a cell below the tile, the lower face of a cell above it =
              // the upper face of its mirrored stencil (bit-identical to the two-sided reconstruction, see recon_hi)
              if (hup) {
                double t = u[0][0]; u[0][0] = u[0][4]; u[0][4] = t;
                t = u[0][1]; u[0][1] = u[0][3]; u[0][3] = t;
              }
              double f = recon_hi<RECON>(G.weno_eps, u[0]);
              if (vr < 2 && !(f > 0.0)) f = u[0][2];   // reading R4: unphysical face values fall back to the cell value
              if (hvalid) {
                if (hup) S.exlo[vr][hr] = f;
                else S.ex[vr][(K == 0) ? hr * EXW : hr] = f;
              }
            }
          }
          if (++st == NS) { st = 0; ph ^= 1u; }
        }
        if (K < 2) {
          bar_states();                                                // A: face states visible
          bar_work();                                                  // C: every Riemann solve has read its states
        }
      }
    }
    return;
  }

  // =================================================================================================
  // compute warps
  // =================================================================================================
  const int tx = tid & (TX - 1), ty = tid / TX;
  const bool in = tx < txn && ty < tyn;
  const int base = ty * EXW + tx;                                      // own flux slot = slot of the left state
  const int hr = lane & 15;                                            // halo unit: row (x) / column (y)
  const bool hup = lane >= 16;                                         //            lower | upper halo cell
  long long c = cell_index(G, i0 + tx, j0 + ty, k0 - 2);
  int st = 0;                                                          // ring stage of the next box to consume
  unsigned ph = 0;                                                     // and its mbarrier phase parity
  // k = k0-2: upper-face z states of plane k0-1; k = k0-1: z flux through the lower face of plane k0
  for (int k = k0 - 2; k < k1; ++k, c += sz) {
#pragma unroll 1
    for (int K = (k < k0) ? 2 : 0; K < 3; ++K) {
      const long long s = G.stride[K];
      const int up = (K == 0) ? 1 : (K == 1) ? EXW : 0;                // own upper-face slot relative to base
      const long long cr = (K == 2) ? c + sz : c, cl = cr - s;         // the face this thread solves
      const bool solve = in && (K < 2 || k >= k0 - 1);
      // ---- a2: reconstruction from the staged boxes, two variables per step so that two independent
      // dependency chains interleave.  fetch(pair): wait for the pair's boxes, read the own stencils into
      // registers, let the pair's halo warp reconstruct the tile's halo cells straight away, and hand the
      // stages back to the producer -- one step BEFORE the own cells of that pair are reconstructed.
      const int own0 = (K == 0) ? ty * (TX + 6) + tx + 3 : (K == 1) ? (ty + 3) * PY + tx + 1 : (2 * TY + ty) * PY + tx + 1;
      const int sst = (K == 0) ? 1 : (K == 1) ? PY : PY * TY;
      const int hal0 = (K == 0) ? hr * (TX + 6) + (hup ? txn + 3 : 2) : (hup ? tyn + 3 : 2) * PY + hr + 1;
      const bool hvalid = hr < ((K == 0) ? tyn : txn);
      const bool edge = in && ((K == 0) ? (tx == txn - 1) : (K == 1) ? (ty == tyn - 1) : false);
      // z: the new upper-face states are parked in this thread's own x slot of the (now idle) exchange buffer
      // -- nobody else touches it between the y phase's last barrier and this thread's next x phase -- and
      // become the carry after the Riemann solve has read the old one
      double* const hi_dst = &S.ex[0][base + ((K == 2) ? 1 : up)];
      const int hi_str = EXP;
      FaceRaw raw;
      double cur[GR][5], nxt[GR][5];
      unsigned rdy[GR];                                                // probe results for the next group's boxes
#pragma unroll
      for (int j = 0; j < GR; ++j) rdy[j] = 0;
      // reconstruct the first cnt (compile-time after unrolling) cells of u, interleaved
      auto recon_n = [&](const double (&u)[GR][5], int cnt, double (&l)[GR], double (&h)[GR]) {
        if (cnt >= GR) {
          recon_cells<RECON, GR>(G.weno_eps, u, l, h);
        } else {
#pragma unroll
          for (int j = 0; j < GR; ++j) {
            if (j < cnt) {
              double l1[1], h1[1];
              const double (&c1)[1][5] = reinterpret_cast<const double (&)[1][5]>(u[j]);
              recon_cells<RECON, 1>(G.weno_eps, c1, l1, h1);
              l[j] = l1[0]; h[j] = h1[0];
            }
          }
        }
      };
      auto fetch = [&](int v0, double (&dst)[GR][5], bool use_probe) {
        const int cnt = (NV - v0 < GR) ? NV - v0 : GR;
        int sj[GR];
#pragma unroll
        for (int j = 0; j < GR; ++j) {
          if (j < cnt) {
            sj[j] = st;
            if (!(use_probe && rdy[j])) mbar_wait(&S.full[st], ph);
            asm volatile("" ::: "memory");                             // no shared-memory load may move above the test
            lds_stencil<RECON>(&S.ring[st][own0], sst, dst[j]);
            if (++st == NS) { st = 0; ph ^= 1u; }
          }
        }
        // The stencils were read through the generic proxy; the refill of this stage is an async-proxy (TMA)
        // write.  Without this cross-proxy fence the refill can overtake the reads: measured on B200 as run-to-run
        // differences in ~0.1 % of the cells (always the last box of a z phase, whose stage is refilled at once).
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) {
#pragma unroll
          for (int j = 0; j < GR; ++j)
            if (j < cnt) mbar_arrive(&S.empty[sj[j]]);
        }
      };
      auto probe = [&](int v0) {                                       // non-blocking probes of the group at (st, ph)
        int s = st;
        unsigned p = ph;
#pragma unroll
        for (int j = 0; j < GR; ++j) {
          rdy[j] = 0;
          if (v0 + j < NV) {
            rdy[j] = mbar_test(&S.full[s], p);
            if (++s == NS) { s = 0; p ^= 1u; }
          }
        }
      };
      fetch(0, cur, false);
      if (GR < NV) probe(GR);
      constexpr int NGRP = (NV + GR - 1) / GR;
      #ifndef RG_PROBE
#define RG_PROBE true
#endif
#ifndef RG_VRAW_BACK
#define RG_VRAW_BACK 2
#endif
      constexpr int VRAW = ((NGRP > RG_VRAW_BACK) ? NGRP - RG_VRAW_BACK : 0) * GR;          // group at which the face metric is fetched
#pragma unroll
      for (int v = 0; v < NV; v += GR) {
        if (v + GR < NV) {
          fetch(v + GR, nxt, RG_PROBE);
          if (v + 2 * GR < NV) probe(v + 2 * GR);
        }
        if (v == VRAW && solve) load_face_raw(T, K, cl, cr, raw);     // consumed after the loop
        {
          double lg[GR], hg[GR];
          recon_n(cur, (NV - v < GR) ? NV - v : GR, lg, hg);
#pragma unroll
          for (int j = 0; j < GR; ++j) {
            if (v + j < NV) {
              const int vr = v + j;
              double l = lg[j], h = hg[j];
              if (vr < 2) {
                if (!(l > 0.0)) l = cur[j][2];
                if (!(h > 0.0)) h = cur[j][2];
              }
              S.los[vr][tid] = l;
              hi_dst[vr * hi_str] = h;
              if (edge) S.exhi[vr][(K == 0) ? ty : tx] = h;
            }
          }
        }
#pragma unroll
        for (int j = 0; j < GR; ++j)
#pragma unroll
          for (int q = 0; q < 5; ++q) cur[j][q] = nxt[j][q];
      }
      if (K < 2) bar_states();                                         // A: face states visible
      // ---- a3: HLLE at the own lower face (x, y) / upper face (z)
      double F[NCONS];
      if (solve) {
#pragma unroll
        for (int q = 0; q < 8; ++q) { pin(raw.l[q]); pin(raw.r[q]); }
        FaceMet m;
        finish_face_met(raw, m);
        // the left states are read from shared memory inside, after the right state's half of the flux
        const double* pl = (K == 2) ? &S.chi[0][tid] : &S.ex[0][base];
        const int pls = (K == 2) ? NT : EXP;
        riemann_mm<CHARGE, NV, WAVE>(G, m, cl, cr, pl, pls, &S.los[0][tid], NT, F);
      }
      if (K < 2) {
        if (solve) {
#pragma unroll
          for (int v = 0; v < NCONS; ++v) S.fx[T.nat[K][v]][base] = F[v];
        }
        bar_work();                                                    // C: fluxes visible
        if (in) {
          const double idx = G.inv_dx[K];
#pragma unroll
          for (int v = 0; v < NCONS; ++v) S.du[v][tid] -= (S.fx[v][base + up] - S.fx[v][base]) * idx;
        }
      } else if (solve) {
        // z: difference against the flux kept from the previous plane, then a5 (divergence part)
        const double idz = G.inv_dx[2], w = (STAGE == 1) ? dt : 0.5 * dt;
        double Fn[NCONS];
#pragma unroll
        for (int v = 0; v < NCONS; ++v) Fn[nat_z(v)] = F[v] * idz;
        if (k >= k0) {
#pragma unroll
          for (int v = 0; v < NCONS; ++v) G.dU[v][c] = w * (S.du[v][tid] - Fn[v]);   // a5 (divergence part), write only
        }
#pragma unroll
        for (int v = 0; v < NCONS; ++v) S.du[v][tid] = Fn[v];          // lower z face of the next plane
      }
      if (K == 2) {                                                    // the parked upper-face states become the carry
#pragma unroll
        for (int vr = 0; vr < NV; ++vr) S.chi[vr][tid] = hi_dst[vr * hi_str];
      }
    }
  }
}

// ---- host side -------------------------------------------------------------------------------------
bool rhs_tma_supported(const GridView& G) {
  // three active directions; TMA needs 16-byte multiples for every global stride (even row pitch)
  return G.n[0] > 1 && G.n[1] > 1 && G.n[2] > 1 && (G.stride[1] % 2) == 0 && (G.stride[2] % 2) == 0;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

// Tensor maps over the 17 equally spaced fields P[0..13], jc[0..2] of the slab, viewed as a 4D tensor
// (x, y, z, field) of doubles; one map per direction (the box shape is part of the map).
void* tma_create(const GridView& G) {
  if (!rhs_tma_supported(G)) return nullptr;
  EncodeTiledFn enc = encode_fn();
  if (!enc) return nullptr;
  const long long fs = G.P[1] - G.P[0];
  for (int v = 1; v < NPRIM; ++v) if (G.P[v] - G.P[v - 1] != fs) return nullptr;
  if (G.jc[0] - G.P[NPRIM - 1] != fs || G.jc[1] - G.jc[0] != fs || G.jc[2] - G.jc[1] != fs) return nullptr;
  TmaMaps* M = new TmaMaps;
  const cuuint64_t dims[4] = {(cuuint64_t)G.np[0], (cuuint64_t)G.np[1], (cuuint64_t)G.np[2], (cuuint64_t)(NPRIM + 3)};
  const cuuint64_t strides[3] = {(cuuint64_t)G.stride[1] * 8, (cuuint64_t)G.stride[2] * 8, (cuuint64_t)fs * 8};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  const cuuint32_t boxes[3][4] = {{TX + 6, TY, 1, 1}, {PY, TY + 6, 1, 1}, {PY, TY, 5, 1}};
  CUtensorMap* maps[3] = {&M->x, &M->y, &M->z};
  for (int K = 0; K < 3; ++K) {
    const CUresult r = enc(maps[K], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void*)G.P[0], dims, strides, boxes[K], estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { delete M; return nullptr; }
  }
  return M;
}

void tma_destroy(void* state) { delete (TmaMaps*)state; }

static int choose_cz(const GridView& G, int sm_count) {
  // one CTA per SM: pick the pencil length that minimises (waves of sm_count CTAs) x (planes per CTA + the two
  // lead-in z phases, ~2/3 of a plane)
  const long long tiles = (long long)((G.n[0] + TX - 1) / TX) * ((G.n[1] + TY - 1) / TY);
  int best = G.n[2];
  double best_cost = 1e300;
  for (int chunks = 1; chunks <= G.n[2] && chunks <= 4096; ++chunks) {
    const int cz = (G.n[2] + chunks - 1) / chunks;
    if (cz < 4 && chunks > 1) break;
    const long long ctas = tiles * ((G.n[2] + cz - 1) / cz);
    const double cost = (double)((ctas + sm_count - 1) / sm_count) * (cz + 0.7);
    if (cost < best_cost) { best_cost = cost; best = cz; }
  }
  return best;
}

template <int RECON, int CHARGE, int STAGE, int WAVE>
static cudaError_t launch_one(const GridView& G, const TmaMaps& M, double dt, int sm_count, cudaStream_t st) {
  const int cz = choose_cz(G, sm_count);
  const PencilTabs T = make_tabs(G);
  dim3 block(NTHREADS, 1, 1);
  dim3 grid((G.n[0] + TX - 1) / TX, (G.n[1] + TY - 1) / TY, (G.n[2] + cz - 1) / cz);
  const size_t smem = sizeof(Smem);
  cudaError_t e = cudaFuncSetAttribute(k_flux_tma<RECON, CHARGE, STAGE, WAVE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_flux_tma<RECON, CHARGE, STAGE, WAVE><<<grid, block, smem, st>>>(G, T, M, dt, cz);
  return cudaGetLastError();
}

template <int RECON, int CHARGE>
static cudaError_t launch_rc(const GridView& G, const TmaMaps& M, double dt, int stage, int sm_count, cudaStream_t st) {
  if (G.wave_mode == WAVE_MHD_INSIDE)
    return stage == 1 ? launch_one<RECON, CHARGE, 1, WAVE_MHD_INSIDE>(G, M, dt, sm_count, st)
                      : launch_one<RECON, CHARGE, 2, WAVE_MHD_INSIDE>(G, M, dt, sm_count, st);
  return stage == 1 ? launch_one<RECON, CHARGE, 1, WAVE_LIGHT>(G, M, dt, sm_count, st)
                    : launch_one<RECON, CHARGE, 2, WAVE_LIGHT>(G, M, dt, sm_count, st);
}

cudaError_t launch_rhs_tma(const GridView& G, const void* state, double dt, int stage, int recon, int sm_count, cudaStream_t st) {
  if (!state) return cudaErrorInvalidValue;
  const TmaMaps& M = *(const TmaMaps*)state;
  const bool ohm = G.charge_mode == CHARGE_FACE_OHM;
  switch (recon) {
    case RECON_MINMOD:
      return ohm ? launch_rc<RECON_MINMOD, CHARGE_FACE_OHM>(G, M, dt, stage, sm_count, st)
                 : launch_rc<RECON_MINMOD, CHARGE_CELL_CURRENT>(G, M, dt, stage, sm_count, st);
    case RECON_MC:
      return ohm ? launch_rc<RECON_MC, CHARGE_FACE_OHM>(G, M, dt, stage, sm_count, st)
                 : launch_rc<RECON_MC, CHARGE_CELL_CURRENT>(G, M, dt, stage, sm_count, st);
    default:
      return ohm ? launch_rc<RECON_WENO5, CHARGE_FACE_OHM>(G, M, dt, stage, sm_count, st)
                 : launch_rc<RECON_WENO5, CHARGE_CELL_CURRENT>(G, M, dt, stage, sm_count, st);
  }
}

}  // namespace rg
