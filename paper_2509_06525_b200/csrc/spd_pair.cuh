// The closed form of a pair's 9x9 s,p,d block (file header of spd9.cu) for the translation units that build
// such blocks: spd9.cu (species tables) and mlp.cu (integrals from MLP_lambda, Eq. 2).  Product code; nothing
// here is used by oracle/.
#pragma once

#include "common.cuh"

namespace gtb {

constexpr int kNc = 14;             // coefficient combinations per ordered species pair
constexpr double kS3 = 1.7320508075688772;   // sqrt(3)
constexpr double kK = 1.1547005383792517;    // 2 / sqrt(3)

// the 14 combinations of the closed form above, from V = sk[si][sj], Vt = sk[sj][si]
// (ss_s, sp_s, pp_s, pp_p, sd_s, pd_s, pd_p, dd_s, dd_p, dd_d)
__host__ __device__ inline void pair_coefficients(const double* V, const double* Vt, double* c) {
  c[0] = V[0];                                        // ss
  c[1] = V[1];                                        // s <- p
  c[2] = V[4];                                        // s <- d
  c[3] = -Vt[1];                                      // p <- s
  c[4] = V[3];                                        // p <- p: delta
  c[5] = V[2] - V[3];                                 //          u u^T
  c[6] = V[5] - kK * V[6];                            // p <- d: u D^T
  c[7] = kK * V[6];                                   //          G^T
  c[8] = Vt[4];                                       // d <- s
  c[9] = -(Vt[5] - kK * Vt[6]);                       // d <- p: D u^T
  c[10] = -kK * Vt[6];                                //          G
  c[11] = V[9];                                       // d <- d: delta
  c[12] = V[7] - 4.0 / 3.0 * V[8] + 1.0 / 3.0 * V[9]; //          D D^T
  c[13] = 4.0 / 3.0 * (V[8] - V[9]);                  //          G G^T
}

struct Geometry {
  double l, m, n;   // bond direction
  double f;         // exp(-beta (r/r0 - 1))
};

// D_a = u^T A_a u, order xy, yz, zx, x2-y2, z2
__device__ __forceinline__ void angular_d(const Geometry& g, double D[5]) {
  D[0] = kS3 * g.l * g.m;
  D[1] = kS3 * g.m * g.n;
  D[2] = kS3 * g.n * g.l;
  D[3] = 0.5 * kS3 * (g.l * g.l - g.m * g.m);
  D[4] = g.n * g.n - 0.5 * (g.l * g.l + g.m * g.m);
}

// G_a = A_a u
__device__ __forceinline__ void angular_g(const Geometry& g, double G[5][3]) {
  const double h = 0.5 * kS3;
  G[0][0] = h * g.m; G[0][1] = h * g.l; G[0][2] = 0.0;
  G[1][0] = 0.0; G[1][1] = h * g.n; G[1][2] = h * g.m;
  G[2][0] = h * g.n; G[2][1] = 0.0; G[2][2] = h * g.l;
  G[3][0] = h * g.l; G[3][1] = -h * g.m; G[3][2] = 0.0;
  G[4][0] = -0.5 * g.l; G[4][1] = -0.5 * g.m; G[4][2] = g.n;
}

// the explicit 9x9 block E[mu][nu] of the pair (closed form in the file header); c already holds f
__device__ inline void pair_block(const Geometry& g, const double* c, double E[9][9]) {
  const double u[3] = {g.l, g.m, g.n};
  double D[5], G[5][3];
  angular_d(g, D);
  angular_g(g, G);
  E[0][0] = c[0];
  for (int b = 0; b < 3; ++b) {
    E[0][1 + b] = c[1] * u[b];
    E[1 + b][0] = c[3] * u[b];
    for (int a = 0; a < 3; ++a) E[1 + a][1 + b] = (a == b ? c[4] : 0.0) + c[5] * u[a] * u[b];
  }
  for (int b = 0; b < 5; ++b) {
    E[0][4 + b] = c[2] * D[b];
    E[4 + b][0] = c[8] * D[b];
    for (int a = 0; a < 3; ++a) {
      E[1 + a][4 + b] = c[6] * u[a] * D[b] + c[7] * G[b][a];
      E[4 + b][1 + a] = c[9] * D[b] * u[a] + c[10] * G[b][a];
    }
    for (int a = 0; a < 5; ++a)
      E[4 + a][4 + b] = (a == b ? c[11] : 0.0) + c[12] * D[a] * D[b] +
                        c[13] * (G[a][0] * G[b][0] + G[a][1] * G[b][1] + G[a][2] * G[b][2]);
  }
}

}  // namespace gtb
