// Internal structures shared by the host plan builder (plan.cpp) and the CUDA side (*.cu).
// Not part of the C ABI (include/gpw.h is).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "gpw.h"

#if defined(__CUDACC__)
#define GPW_CX __host__ __device__ constexpr
#else
#define GPW_CX constexpr
#endif

namespace gpw {

constexpr int MAXL = GPW_MAX_L;          // shells up to f
constexpr int MAXLP = 2 * MAXL;          // pair polynomial degree L = la + lb <= 6
constexpr int NLSEG = MAXLP + 1;         // visit lists are segmented by L = 0..6
// Degree offsets: the grid kernels evaluate a pair polynomial (or accumulate pair moments) of degree L + off.
//   off 0: density / potential (Eq. 3-4);  off 1: nuclear gradient (Alg. 3: one derivative of one function);
//   off 2: kinetic-energy density tau and its potential (Eq. 15-16: one derivative of each function)
constexpr int NOFF = 3;
constexpr int MAXDEG = MAXLP + NOFF - 1; // largest polynomial degree, 8
constexpr int TILE = 4;                  // grid block edge
// integration stages bricks of BR1 x BR2 x BR3 grid blocks in shared memory; one block thick along n1 so
// that a lane (which owns one n1 plane of a block) keeps the same u1 for every block of a brick entry
constexpr int BR1 = 1, BR2 = 5, BR3 = 5;
constexpr int BRICK_TILES = BR1 * BR2 * BR3;
static_assert(BR1 == 1 && BRICK_TILES <= 32, "brick: one block along n1, mask of at most 32 blocks");

// number of monomials u1^kx u2^ky u3^kz with kx+ky+kz <= L
GPW_CX int ncoef(int L) { return (L + 1) * (L + 2) * (L + 3) / 6; }
// per-pair workspace stride (kept even so that rows stay 16-byte aligned)
GPW_CX int ncoef_pad(int L) { return (ncoef(L) + 1) & ~1; }
GPW_CX int ncart(int l) { return (l + 1) * (l + 2) / 2; }

// Geometry of one multigrid level (plain data: copied to the device as is).
struct LevelGeom {
    int N[3];        // mesh
    int T[3];        // 4x4x4 blocks per axis
    int ntile;       // T[0]*T[1]*T[2]
    int nbrick;      // B[0]*B[1]*B[2]
    int B[3];        // bricks per axis, ceil(T_i / BR_i) (the last brick of an axis may be ragged)
    int pad0;
    double H[9];     // H[c*3+i] = component c of the grid step vector a_i / N_i :  r - P = H (n - n_P)
    double Hinv[9];  // Hinv[i*3+c]:  u_i = sum_c Hinv[i*3+c] X_c
    double Gm[6];    // H^T H, packed 11 22 33 12 13 23 : |H u|^2 = u^T Gm u
    double dV;       // Omega / (N1 N2 N3)   (Eq. 29)
    double ecut;     // E_alpha of T5
};

// Pair record read by the collocation / integration kernels (64 bytes, four 16-byte loads).
struct TaskK {
    double nP[3];        // Gaussian-product centre P in grid-index units of its level
    double ap;           // a_p = a_a + a_b
    double c22, c23;     // exp(-2 a_p Gm22), exp(-2 a_p Gm23): second-order ratios of the Gaussian recursion
    double c33;          // exp(-2 a_p Gm33)   (Eq. 25; the cross term is the integer-index reading of A.31-A.32)
    long long coef_off;  // offset (doubles) of the pair's polynomial / moment vector in the degree-L workspace
};
static_assert(sizeof(TaskK) == 64, "TaskK must be 64 bytes");

// Pair record read by the pre-pass (D block -> polynomial) and post-pass (moments -> F block).
struct TaskP {
    double PA[3];    // P - A
    double PB[3];    // P - (B + T)
    double pref;     // coef_a coef_b exp(-a_a a_b / a_p |A - B - T|^2)
    double aa, ab;   // the two primitive exponents (derivative variants: Eq. 15-16, Alg. 3)
    int ao_a, ao_b;
    int atom_a, atom_b;
    short la, lb;
    short level;
    short sym;       // 1: use D_ab + D_ba and mirror F (hermi, not the a==b,T==0 pair)
};
static_assert(sizeof(TaskP) == 96, "TaskP must be 96 bytes");

// One (pair, 4x4x4 block) visit in a block's list.
struct Visit {
    int task;             // global pair index
    signed char s[3];     // lattice wraps: unwrapped block = stored block + s * T
    unsigned char pad;
};
static_assert(sizeof(Visit) == 8, "Visit must be 8 bytes");

// Work item of the grid kernels: a contiguous range of one block's visit list.
struct Item {
    int level;
    int tile;             // stored block index on its level
    unsigned lo, hi;      // visit range relative to the block's list
    int single;           // 1: the only item of its block (plain store), 0: accumulate atomically
    int pad;
    long long vstart;     // index of the item's first visit in the plan's visit list (= tile_base of the block + lo):
                          // saves the collocation warp one dependent load at its start
};
static_assert(sizeof(Item) == 32, "Item must be 32 bytes");

// One (pair, lattice image, brick) entry of a brick's list: which of the brick's blocks the pair visits.
struct BEntry {
    int task;
    signed char s[3];     // lattice wraps of this image
    unsigned char L;      // la + lb
    unsigned mask;        // bit (t2*BR3 + t3) set: block (t2,t3) of the brick is visited
    unsigned pad;
};
static_assert(sizeof(BEntry) == 16, "BEntry must be 16 bytes");

// Work item of the integration kernel: a range of one brick's entry list.
struct BItem {
    int level;
    int brick;
    long long base;       // global index of the brick's first entry
    unsigned lo, hi;      // entry range relative to the brick's list
    unsigned seg[8];      // start of each L segment of the brick's list (relative); seg[7] = list length
    unsigned pad[2];
};
static_assert(sizeof(BItem) == 64, "BItem must be 64 bytes");

// One primitive as the device pair screen reads it (T1 radius from the host).
struct DevPrim {
    double A[3];     // centre
    double exp, coef, rad;
    int shl, l, ao, atom;
};

struct HostTask {
    int shl_a, prim_a, shl_b, prim_b;
    int T[3];
    int level, la, lb;
    double R, ap, pref;
    double P[3], A[3], Bt[3];
    int sym;
};

struct HostPlan {
    // inputs kept
    double cell[9], binv[9], bnorm[3], omega;
    int natm = 0, nshl = 0, nprim = 0, nlevel = 0, nao = 0, hermi = 0;
    double tau = 0, rel_cutoff = 0;
    std::vector<int> ao_loc;
    std::vector<LevelGeom> lev;
    std::vector<std::vector<double>> S;   // per level: Cartesian -> grid-index monomial maps, degree blocks
    std::vector<DevPrim> prims;           // every primitive with its radius (T1)
    long ntask = 0;                       // kept pairs (= task.size() once the host holds them)
    std::vector<HostTask> task;           // sorted by (level, L, la, enumeration order); with a device the pairs are
                                          // screened there (pairs_device.cu) and this stays empty
    std::vector<TaskK> taskK;
    std::vector<TaskP> taskP;
    // per degree offset `off`: workspace offset of pair i (global index) of class (level, L)
    //   = coef_base[off][level][L] + i * ncoef_pad(L + off);   ncoef_total[off] doubles in all
    long long ncoef_total[NOFF] = {0};
    long long coef_base[NOFF][GPW_MAX_LEVEL][NLSEG + 1] = {{{0}}};
    // per level block lists
    std::vector<std::vector<long long>> tile_base;   // [level][ntile+1] global visit index
    std::vector<std::vector<unsigned>> seg;          // [level][ntile*8] start of each L segment (relative)
    std::vector<Visit> visit;                        // all levels, level-major, block-major
    std::vector<Item> item;                          // sorted by descending size
    std::vector<std::vector<long long>> brick_base;  // [level][nbrick+1] global entry index
    std::vector<BEntry> bentry;                      // all levels, level-major, brick-major; inside a brick by L,
                                                     // inside an L segment by decreasing number of visited blocks
    std::vector<BItem> bitem;                        // sorted by descending work
    long nitem = 0, nbitem = 0;                      // work items of the two grid kernels
    long long nvisit_total = 0;
    double circ[GPW_MAX_LEVEL] = {0};                // circumradius of a 4x4x4 block about its centre, per level
    int max_L = 0;                                   // largest la + lb present
    long big_lo[GPW_MAX_LEVEL] = {0}, big_hi[GPW_MAX_LEVEL] = {0};   // per level, the pairs with la + lb >= 5 (contiguous: the
                                                     // last classes of the level in the sort order)
    bool ortho = false;                              // the lattice vectors are mutually orthogonal (every Gm diagonal)
    bool hdiag = false;                              // ... and along the Cartesian axes (every H, hence every S_d, diagonal)
    int max_l = 0;                                   // largest shell angular momentum
    long nvisit_level[GPW_MAX_LEVEL] = {0};
    long ntask_level[GPW_MAX_LEVEL] = {0};
    long nvisit_class[GPW_MAX_LEVEL][MAXL + 1][MAXL + 1] = {{{0}}};
    double build_seconds = 0;
};

// offsets of the degree blocks inside S[level]: block d is n_d x n_d, n_d = (d+1)(d+2)/2
GPW_CX int s_block_off(int d) {
    int o = 0;
    for (int e = 0; e < d; e++) { int n = (e + 1) * (e + 2) / 2; o += n * n; }
    return o;
}
constexpr int S_TOTAL = s_block_off(MAXDEG + 1);   // degree blocks 0..8: 4917 doubles

void set_error(const std::string &msg);

// plan.cpp
int build_host_plan(const double *cell, int natm, const double *xyz, int nshl, const int *shl_atom,
                    const int *shl_l, const int *shl_nprim, const int *shl_prim_off,
                    const double *prim_exp, const double *prim_coef, int nlevel, const int *mesh,
                    double tau, double rel_cutoff, int hermi, bool on_host, HostPlan **out);

}  // namespace gpw
