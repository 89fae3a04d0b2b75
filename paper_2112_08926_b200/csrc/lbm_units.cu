// lbm_units.cu -- table of the (velocity set, storage format) units compiled from lbm_unit.cu (formats 0-6) and lbm_unit64.cu (7, 8).
#include "lbm_internal.h"

namespace lbmk {

#define LBM_DECL(q, f) extern const UnitOps lbm_unit_q##q##_f##f;
#define LBM_DECL_Q(q) LBM_DECL(q, 0) LBM_DECL(q, 1) LBM_DECL(q, 2) LBM_DECL(q, 3) LBM_DECL(q, 4) LBM_DECL(q, 5) LBM_DECL(q, 6) LBM_DECL(q, 7) LBM_DECL(q, 8)
LBM_DECL_Q(9)
LBM_DECL_Q(19)
LBM_DECL_Q(27)

#define LBM_ROW(q) {&lbm_unit_q##q##_f0, &lbm_unit_q##q##_f1, &lbm_unit_q##q##_f2, &lbm_unit_q##q##_f3, \
                    &lbm_unit_q##q##_f4, &lbm_unit_q##q##_f5, &lbm_unit_q##q##_f6, \
                    &lbm_unit_q##q##_f7, &lbm_unit_q##q##_f8}

const UnitOps *unit_ops(int q, int fmt) {
    static const UnitOps *const table[3][9] = {LBM_ROW(9), LBM_ROW(19), LBM_ROW(27)};
    if (fmt < 0 || fmt > 8) return nullptr;
    const int row = q == 9 ? 0 : q == 19 ? 1 : q == 27 ? 2 : -1;
    return row < 0 ? nullptr : table[row][fmt];
}

}  // namespace lbmk
