// lbm_units.cu -- table of the (velocity set, storage format) units compiled from lbm_unit.cu.
#include "lbm_internal.h"

namespace lbmk {

#define LBM_DECL(q, f) extern const UnitOps lbm_unit_q##q##_f##f;
#define LBM_DECL_Q(q) LBM_DECL(q, 0) LBM_DECL(q, 1) LBM_DECL(q, 2) LBM_DECL(q, 3) LBM_DECL(q, 4) LBM_DECL(q, 5) LBM_DECL(q, 6)
LBM_DECL_Q(9)
LBM_DECL_Q(19)
LBM_DECL_Q(27)

#define LBM_ROW(q) {&lbm_unit_q##q##_f0, &lbm_unit_q##q##_f1, &lbm_unit_q##q##_f2, &lbm_unit_q##q##_f3, \
                    &lbm_unit_q##q##_f4, &lbm_unit_q##q##_f5, &lbm_unit_q##q##_f6}

const UnitOps *unit_ops(int q, int fmt) {
    static const UnitOps *const table[3][7] = {LBM_ROW(9), LBM_ROW(19), LBM_ROW(27)};
    if (fmt < 0 || fmt > 6) return nullptr;
    const int row = q == 9 ? 0 : q == 19 ? 1 : q == 27 ? 2 : -1;
    return row < 0 ? nullptr : table[row][fmt];
}

}  // namespace lbmk
