// Closed-form entries of the spatial base matrices on the g x g grid (BASELINE.json configs[0];
// readings R3, R21): C = h^2 I, G = 5-point graph Laplacian (degree - adjacency), K2 = G C^-1 G.
// Term c of the prior pairs temporal M_c with spatial K_c:  c=0: K2,  c=1: G,  c=2: C.
#pragma once

__device__ __forceinline__ double st_G(int g, int y, int x, int y2, int x2) {
  const int ad = abs(y2 - y) + abs(x2 - x);
  if (ad == 0) return (double)((x > 0) + (x < g - 1) + (y > 0) + (y < g - 1));
  return ad == 1 ? -1.0 : 0.0;
}

__device__ __forceinline__ double st_K2(int g, double inv_h2, int y, int x, int y2, int x2) {
  if (abs(y2 - y) + abs(x2 - x) > 2) return 0.0;
  double s = st_G(g, y, x, y, x) * st_G(g, y, x, y2, x2);  // u = s itself
  if (x > 0) s -= st_G(g, y, x - 1, y2, x2);               // G[s][u] = -1 for each neighbour u
  if (x < g - 1) s -= st_G(g, y, x + 1, y2, x2);
  if (y > 0) s -= st_G(g, y - 1, x, y2, x2);
  if (y < g - 1) s -= st_G(g, y + 1, x, y2, x2);
  return s * inv_h2;
}

// K_c[s][s2] for all three terms at once
__device__ __forceinline__ void st_K(int g, double h, int y, int x, int y2, int x2, double kv[3]) {
  kv[0] = st_K2(g, 1.0 / (h * h), y, x, y2, x2);
  kv[1] = st_G(g, y, x, y2, x2);
  kv[2] = (y == y2 && x == x2) ? h * h : 0.0;
}

// Temporal weights (reading R4): diagonal of M_c at time t, and the (t+1, t) entry.
__device__ __forceinline__ void st_Mdiag(int nt, int t, double md[3]) {
  md[0] = 1.0;
  md[1] = (nt == 1) ? 0.0 : ((t == 0 || t == nt - 1) ? 1.0 : 2.0);
  md[2] = 2.0;
}
__device__ __forceinline__ void st_Moff(double mo[3]) {
  mo[0] = 0.0;
  mo[1] = -1.0;
  mo[2] = -1.0;
}
