// transport.cu -- explicit M1 transport on the coarse block.
//
// U = (N, F), flux F~ = (F, c^2 P), Eq. 30 (conservative update) with the Lax-Friedrichs /
// GLF interface flux Eq. 32, unsplit over the three directions (A4), closure Eq. 22-23 (A1, A2), reduced speed
// of light everywhere (A3), boundary conditions of PAPER.md:436 (A13).
//
// In the internal variables phi = F / c the own-cell flux cancels and the whole update is
//     U' = (1 - 3 nu) U + (nu/2) sum_d [ (U - G_d)(i+e_d) + (U + G_d)(i-e_d) ],     nu = c dt / dx,
//     G_d = (phi_d, Pi_dx, Pi_dy, Pi_dz),   Pi = P (in units of N) = a I + b phi(x)phi,
//     a = N (1/3 - q),  b = 3 q / (N f^2),  q = f^2 / (2 + sqrt(4 - 3 f^2)),  f = |phi| / N clipped to 1
// (algebraically Levermore's chi = 1/3 + 2q; the form avoids the cancellation of 3 chi - 1 at small f).
// Each cell's closure (a, b) is computed ONCE, by the thread that owns the cell (or its halo copy), and staged in
// shared memory next to U; the paper's own stencil-array design recomputes it for every neighbour.
//
// Kernel shape: 2.5-D streaming.  A CTA owns a TX x TY column of cells and marches along z through a chunk of
// planes; z-neighbours live in registers, x/y-neighbours come from a double-buffered shared-memory plane
// (one barrier per plane).  Loads of plane k+2 are issued while plane k is computed.  HBM traffic is the
// algorithmic 16 B read + 16 B write per cell-group plus the tile-edge halo (served from L2).
#include "emma_rt_internal.cuh"

namespace emma {

namespace {

constexpr int TX = 32, TY = 16;
constexpr int SW = TX + 2;                     // shared plane width incl. halo
constexpr int SH = TY + 2;

__device__ __forceinline__ void closure_ab(float N, float px, float py, float pz, float& a, float& b)
{
  // A2: N <= 0 -> f = 0.  A denormal N (light that has just reached a dark cell) counts as 0: rcp.ftz of it is inf.
  float rN = (N >= 1.1754944e-38f) ? frcp(N) : 0.f;
  float rx = px * rN, ry = py * rN, rz = pz * rN;
  float f2raw = rx * rx + ry * ry + rz * rz;
  float f2 = fminf(f2raw, 1.f);                // A2: f clipped to [0,1]
  float s = fsqrt(4.f - 3.f * f2);
  float q = f2 * frcp(2.f + s);
  a = N * (0.33333334f - q);
  // A1: |F| = 0 -> no n(x)n term; below f^2 = 1e-30 the term (<= f^2 N) is far under fp32 resolution of a
  b = (f2raw > 1e-30f) ? 3.f * q * rN * frcp(f2raw) : 0.f;
}

// map an index that may be one cell outside [0,n) through the boundary condition of that face (A13)
__device__ __forceinline__ int bc_map(int i, int n, int bc_lo, int bc_hi, bool& flip)
{
  flip = false;
  if (i < 0) {
    if (bc_lo == EMMA_RT_BC_PERIODIC) return i + n;
    flip = (bc_lo == EMMA_RT_BC_REFLECTIVE);
    return 0;
  }
  if (i >= n) {
    if (bc_hi == EMMA_RT_BC_PERIODIC) return i - n;
    flip = (bc_hi == EMMA_RT_BC_REFLECTIVE);
    return n - 1;
  }
  return i;
}

// contribution of the neighbour on the + side of direction d:  U - G_d
template <int D>
__device__ __forceinline__ void add_plus(float4& acc, const float4& U, float a, float b)
{
  float pd = (D == 0) ? U.y : (D == 1) ? U.z : U.w;
  float u = 1.f - b * pd;
  acc.x += U.x - pd;
  acc.y = fmaf(U.y, u, acc.y);
  acc.z = fmaf(U.z, u, acc.z);
  acc.w = fmaf(U.w, u, acc.w);
  if (D == 0) acc.y -= a; else if (D == 1) acc.z -= a; else acc.w -= a;
}
// neighbour on the - side:  U + G_d
template <int D>
__device__ __forceinline__ void add_minus(float4& acc, const float4& U, float a, float b)
{
  float pd = (D == 0) ? U.y : (D == 1) ? U.z : U.w;
  float u = 1.f + b * pd;
  acc.x += U.x + pd;
  acc.y = fmaf(U.y, u, acc.y);
  acc.z = fmaf(U.z, u, acc.z);
  acc.w = fmaf(U.w, u, acc.w);
  if (D == 0) acc.y += a; else if (D == 1) acc.z += a; else acc.w += a;
}

__global__ void __launch_bounds__(TX* TY, 2)
transport_kernel(const TransportParams p, const float4* __restrict__ Uin, float4* __restrict__ Uout,
                 Partial* __restrict__ parts)
{
  __shared__ float4 sU[2][SH][SW];
  __shared__ float2 sAB[2][SH][SW];

  const int n = p.n;
  // block -> (tile x, tile y, z chunk, group), tile x fastest so that concurrently resident CTAs are neighbours
  int bid = blockIdx.x;
  const int tix = bid % p.tiles_x; bid /= p.tiles_x;
  const int tiy = bid % p.tiles_y; bid /= p.tiles_y;
  const int izc = bid % p.nzc;     bid /= p.nzc;
  const int g = bid;
  const int tx = threadIdx.x % TX, ty = threadIdx.x / TX;
  const int x0 = tix * TX, y0 = tiy * TY;
  const int wx = min(TX, n - x0), wy = min(TY, n - y0);
  const int z0 = izc * p.zchunk, z1 = min(n, z0 + p.zchunk);
  const bool active = (tx < wx) && (ty < wy);
  const int x = x0 + tx, y = y0 + ty;
  const size_t plane = (size_t)n * n;
  const float4* __restrict__ Ug = Uin + (size_t)g * plane * n;
  float4* __restrict__ Vg = Uout + (size_t)g * plane * n;
  const size_t col = active ? ((size_t)y * n + x) : 0;

  // halo duty: thread t < 2*wy + 2*wx also stages one halo cell per plane
  const int t = threadIdx.x;
  const bool hduty = t < 2 * wy + 2 * wx;
  int hsx = 0, hsy = 0, hflipc = 0;            // shared coords of my halo cell; component to flip (1..2) or 0
  size_t hcol = 0;
  if (hduty) {
    bool fl;
    if (t < 2 * wy) {                          // left / right columns
      const int r = (t < wy) ? t : t - wy;
      const int gx = bc_map((t < wy) ? x0 - 1 : x0 + wx, n, p.bc[0], p.bc[1], fl);
      hsx = (t < wy) ? 0 : wx + 1; hsy = r + 1;
      hcol = (size_t)(y0 + r) * n + gx;
      hflipc = fl ? 1 : 0;
    } else {                                   // bottom / top rows
      const int q = t - 2 * wy;
      const int r = (q < wx) ? q : q - wx;
      const int gy = bc_map((q < wx) ? y0 - 1 : y0 + wy, n, p.bc[2], p.bc[3], fl);
      hsx = r + 1; hsy = (q < wx) ? 0 : wy + 1;
      hcol = (size_t)gy * n + (x0 + r);
      hflipc = fl ? 2 : 0;
    }
  }

  const float nu = p.nu, c0 = p.c0, c1 = p.c1;
  Acc acc_d;

  // ---- prologue: planes z0-1 (-> Wm), z0 (-> cur), z0+1 (-> raw next); halo of z0, z0+1
  bool flz;
  float4 Wm = make_float4(0, 0, 0, 0);
  float4 cur = make_float4(0, 0, 0, 0), nxt = make_float4(0, 0, 0, 0), hcur = make_float4(0, 0, 0, 0),
         hnxt = make_float4(0, 0, 0, 0);
  float ca = 0, cb = 0;
  bool nxt_flip = false;
  {
    const int zm = bc_map(z0 - 1, n, p.bc[4], p.bc[5], flz);
    if (active) {
      float4 pm = __ldg(Ug + (size_t)zm * plane + col);
      if (flz) pm.w = -pm.w;
      float a, b;
      closure_ab(pm.x, pm.y, pm.z, pm.w, a, b);
      add_minus<2>(Wm, pm, a, b);              // Wm = U + G_z of the plane below
      cur = __ldg(Ug + (size_t)z0 * plane + col);
      closure_ab(cur.x, cur.y, cur.z, cur.w, ca, cb);
    }
    if (hduty) hcur = __ldg(Ug + (size_t)z0 * plane + hcol);
    const int zn = bc_map(z0 + 1, n, p.bc[4], p.bc[5], nxt_flip);
    if (active) nxt = __ldg(Ug + (size_t)zn * plane + col);
    if (hduty && z0 + 1 < z1) hnxt = __ldg(Ug + (size_t)(z0 + 1) * plane + hcol);
  }

  for (int z = z0; z < z1; z++) {
    const int buf = z & 1;
    // (a) stage this plane: own cell and halo cell, each with its closure
    if (active) {
      sU[buf][ty + 1][tx + 1] = cur;
      sAB[buf][ty + 1][tx + 1] = make_float2(ca, cb);
    }
    if (hduty) {
      float4 h = hcur;
      if (hflipc == 1) h.y = -h.y; else if (hflipc == 2) h.z = -h.z;
      float a, b;
      closure_ab(h.x, h.y, h.z, h.w, a, b);
      sU[buf][hsy][hsx] = h;
      sAB[buf][hsy][hsx] = make_float2(a, b);
    }
    // (b) issue the loads of plane z+2 (consumed two iterations from now)
    float4 nn = make_float4(0, 0, 0, 0), hnn = make_float4(0, 0, 0, 0);
    bool nn_flip = false;
    if (z + 1 < z1) {
      const int z2 = bc_map(z + 2, n, p.bc[4], p.bc[5], nn_flip);
      if (active) nn = __ldg(Ug + (size_t)z2 * plane + col);
      if (hduty && z + 2 < z1) hnn = __ldg(Ug + (size_t)(z + 2) * plane + hcol);
    }
    // (c) closure of the plane above and its contribution U - G_z
    float4 acc = Wm;
    float na = 0, nb = 0;
    float4 nx = nxt;
    if (active) {
      if (nxt_flip) nx.w = -nx.w;
      closure_ab(nx.x, nx.y, nx.z, nx.w, na, nb);
      add_plus<2>(acc, nx, na, nb);
    }
    __syncthreads();
    // (d) x / y neighbours from shared memory
    if (active) {
      {
        const float4 u = sU[buf][ty + 1][tx]; const float2 ab = sAB[buf][ty + 1][tx];
        add_minus<0>(acc, u, ab.x, ab.y);
      }
      {
        const float4 u = sU[buf][ty + 1][tx + 2]; const float2 ab = sAB[buf][ty + 1][tx + 2];
        add_plus<0>(acc, u, ab.x, ab.y);
      }
      {
        const float4 u = sU[buf][ty][tx + 1]; const float2 ab = sAB[buf][ty][tx + 1];
        add_minus<1>(acc, u, ab.x, ab.y);
      }
      {
        const float4 u = sU[buf][ty + 2][tx + 1]; const float2 ab = sAB[buf][ty + 2][tx + 1];
        add_plus<1>(acc, u, ab.x, ab.y);
      }
      float4 o;
      o.x = fmaf(c1, acc.x, c0 * cur.x);
      o.y = fmaf(c1, acc.y, c0 * cur.y);
      o.z = fmaf(c1, acc.z, c0 * cur.z);
      o.w = fmaf(c1, acc.w, c0 * cur.w);
      Vg[(size_t)z * plane + col] = o;
      // diagnostics: non-finite scan; N dV total when chemistry is off; outflow through open faces (A15):
      // transmissive face flux = own F_d (ghost copies the cell), reflective face flux = 0
      if (!(fabsf(o.x) + fabsf(o.y) + fabsf(o.z) + fabsf(o.w) < __int_as_float(0x7f800000))) acc_d.nonfinite++;
      if (p.want_total) acc_d.total += (double)o.x;
      if (x == 0 && p.bc[0] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)cur.y;
      if (x == n - 1 && p.bc[1] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cur.y;
      if (y == 0 && p.bc[2] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)cur.z;
      if (y == n - 1 && p.bc[3] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cur.z;
      if (z == 0 && p.bc[4] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow -= (double)cur.w;
      if (z == n - 1 && p.bc[5] == EMMA_RT_BC_TRANSMISSIVE) acc_d.outflow += (double)cur.w;
      // (e) rotate the z pipeline: this plane becomes the one below
      Wm = make_float4(0, 0, 0, 0);
      add_minus<2>(Wm, cur, ca, cb);
      cur = nx; ca = na; cb = nb;
    }
    nxt = nn; nxt_flip = nn_flip;
    hcur = hnxt; hnxt = hnn;
  }

  // photons: sums are in units of N; scale by nu dV (outflow = c phi dt dx^2 = nu phi dV) resp. dV
  acc_d.outflow *= (double)nu * p.dV;
  acc_d.total *= p.dV;
  block_reduce_store(acc_d, parts + blockIdx.x);
}

}  // namespace

int launch_transport(const TransportParams& p, const float4* Uin, float4* Uout, Partial* parts, int* n_parts,
                     cudaStream_t st)
{
  const int nblk = p.tiles_x * p.tiles_y * p.nzc * p.G;
  transport_kernel<<<nblk, TX * TY, 0, st>>>(p, Uin, Uout, parts);
  *n_parts = nblk;
  return 1;
}

}  // namespace emma
