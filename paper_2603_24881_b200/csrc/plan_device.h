// Interface of the device list builder (plan_device.cu) used by gpw_api.cu.  Not part of the C ABI.
#pragma once
#include "gpw_internal.h"

namespace gpw {

// What the list builder needs of a pair (48 bytes).
struct DevTask {
    double P[3];     // Gaussian-product centre (Cartesian, Bohr)
    double R;        // pair radius R_t (T4)
    int level, L, la, lb;
};

struct LevelList {
    int N[3], T[3], B[3];
    int ntile, nbrick;
    long long tile0, brick0;   // first global block / brick id of the level
};

struct ListGeom {
    double cell[9], binv[9], bnorm[3];
    double circ[GPW_MAX_LEVEL];
    int nlevel, pad;
    LevelList lev[GPW_MAX_LEVEL];
};

// Device arrays written by build_device_lists (owned by the caller afterwards; free with free_device_lists).
struct DeviceLists {
    Visit *visit = nullptr;              // [nvisit] block-major, inside a block by L then pair
    long long nvisit = 0;
    long long *tile_base = nullptr;      // [ntile_all + 1] global visit index of every block's list (levels back to back)
    unsigned *seg = nullptr;             // [ntile_all * 8] start of each L segment relative to the block's list
    Item *item = nullptr;
    long nitem = 0;
    Item *item_hi = nullptr;             // items over the visits of the classes L >= 5 only (second collocation launch of
    long nitem_hi = 0;                   // plans with f shells): the blocks that have such visits, nothing else
    BEntry *bentry = nullptr;            // [nentry] brick-major, inside a brick by L then by decreasing blocks
    long long nentry = 0;
    long long *brick_base = nullptr;     // [nbrick_all + 1]
    BItem *bitem = nullptr;
    long nbitem = 0;
    unsigned long long cls[GPW_MAX_LEVEL][MAXL + 1][MAXL + 1] = {{{0}}};   // visits per (level, la, lb)
    long bytes = 0;
    double seconds = 0;
};

// One kept pair in enumeration order (pairs_device.cu, between its fill and record passes).
struct RawPair {
    int pa, pb, T[3], level;
    double R, ap, pref;
    double P[3], Bt[3];
    int sym, pad;
};

// Device arrays written by build_device_pairs (owned by the caller afterwards; free with free_device_pairs).
struct DevicePairs {
    TaskK *taskK = nullptr;
    TaskP *taskP = nullptr;
    DevTask *devtask = nullptr;      // what the list builder reads; freed by the caller after build_device_lists
    gpw_task *exported = nullptr;    // what gpw_plan_export_tasks copies back
    long ntask = 0;
    long bytes = 0;
};

// Pair screening on the device (T2-T5); fills hp->ntask, coef_base, ncoef_total, ntask_level, max_L.
int build_device_pairs(HostPlan *hp, DevicePairs *out);
void free_device_pairs(DevicePairs *d);

// returns a gpw_status; on failure the message is in gpw_last_error() and nothing is left allocated
// d_task: the ntask pairs on the device, sorted by (level, L)
int build_device_lists(const HostPlan *hp, const DevTask *d_task, int ntask, DeviceLists *out);
void free_device_lists(DeviceLists *l);

}  // namespace gpw
