// Level schedule and tile decode of the time-parallel Phi scan (shared by the SIMT and tcgen05 kernels).
//
// Steps are 0 .. NS-1 with NS = T-1; Phi(t,s) covers steps s .. t-1.  Level 0 is Phi(s+1,s) = A_s.  At level
// l >= 1 the steps are cut into aligned segments [kS, min((k+1)S, NS)) of S = 2^l steps with midpoint
// mid = kS + S/2; every segment whose midpoint is < NS forms all Phi(t,s) = Phi(t,mid) Phi(mid,s) with
// kS <= s < mid < t <= hi.  Both factors lie inside one half-segment, so they were produced at a level < l
// ("forward parallel associative scan", applied to the all-pairs triangular output).
//
// COLUMN_PACKED storage: block (t,s) at index colbase(s) + (t-s-1); for fixed s the blocks t = s+1 .. T-1
// form one contiguous tall row-major matrix, so the stacked left operand [Phi(mid+1,mid); ..; Phi(hi,mid)]
// and each output column [Phi(mid+1,s); ..; Phi(hi,s)] are plain (cnt_t * n) x n matrices.
#pragma once
#include <cstdint>

namespace ltv {

__host__ __device__ inline long long phi_colbase(int T, int s) {
  return static_cast<long long>(s) * (T - 1) - static_cast<long long>(s) * (s - 1) / 2;
}

struct PhiGeom {
  int batch, T, n, P;
  int nc;            // columns per block = row stride of Phi (n, or n + padded p with the observer's PhiY columns)
  int level, S, H;   // segment length, half length (= number of s per segment)
  int nseg;          // segments at this level
  int tm, tn;        // tile sizes
  int NT;            // n-tiles per block column
  int MtF, MtL;      // m-tiles of a full / of the last segment
  int tilesF, tilesL, tilesItem;
  long long total;
};

__host__ __device__ inline PhiGeom phi_geom(int batch, int T, int n, int nc, int level, int tm, int tn) {
  PhiGeom g;
  g.batch = batch; g.T = T; g.n = n; g.nc = nc; g.P = T * (T - 1) / 2;
  g.level = level; g.S = 1 << level; g.H = g.S >> 1;
  const int NS = T - 1;
  g.nseg = (NS > g.H) ? (NS - g.H + g.S - 1) / g.S : 0;
  g.tm = tm; g.tn = tn;
  g.NT = (nc + tn - 1) / tn;
  g.MtF = (g.H * n + tm - 1) / tm;
  int cntL = 0;
  if (g.nseg > 0) {
    const int lo = (g.nseg - 1) * g.S, mid = lo + g.H;
    const int hi = (lo + g.S < NS) ? lo + g.S : NS;
    cntL = hi - mid;
  }
  g.MtL = (cntL * n + tm - 1) / tm;
  g.tilesF = g.MtF * g.H * g.NT;
  g.tilesL = g.MtL * g.H * g.NT;
  g.tilesItem = (g.nseg > 0) ? (g.nseg - 1) * g.tilesF + g.tilesL : 0;
  g.total = static_cast<long long>(g.tilesItem) * batch;
  return g;
}

struct PhiTile {
  int b, s, mid, cnt_t;   // output column s, split node mid, number of t (t = mid+1 .. mid+cnt_t)
  int m_tile, n_tile;
};

// consecutive tile indices share (b, s, n_tile) and walk m_tile: concurrently running CTAs re-use the same
// right-operand tile out of L2
__host__ __device__ inline PhiTile phi_decode(const PhiGeom& g, long long idx) {
  PhiTile t;
  t.b = static_cast<int>(idx / g.tilesItem);
  int rem = static_cast<int>(idx - static_cast<long long>(t.b) * g.tilesItem);
  int k, Mt;
  if (rem < (g.nseg - 1) * g.tilesF) {
    k = rem / g.tilesF;
    rem -= k * g.tilesF;
    Mt = g.MtF;
  } else {
    k = g.nseg - 1;
    rem -= k * g.tilesF;
    Mt = g.MtL;
  }
  const int lo = k * g.S;
  t.mid = lo + g.H;
  const int NS = g.T - 1;
  const int hi = (lo + g.S < NS) ? lo + g.S : NS;
  t.cnt_t = hi - t.mid;
  t.m_tile = rem % Mt;
  rem /= Mt;
  t.n_tile = rem % g.NT;
  t.s = lo + rem / g.NT;
  return t;
}

}  // namespace ltv
