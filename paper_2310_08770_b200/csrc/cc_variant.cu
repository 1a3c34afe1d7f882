// cc_variant.cu -- one translation unit per kernel variant; build.py defines
// CCV_NAME and the template arguments on the nvcc command line.
#include "cc_fused.cuh"

using VariantCfg = ccf::Cfg<CCV_H, CCV_W, CCV_CS, CCV_PIX, CCV_NT, CCV_TM1, CCV_TN1, CCV_TM2, CCV_TN2, CCV_SG, CCV_BK1, CCV_G2,
                            CCV_R2, CCV_KS2, CCV_NSTG, CCV_PFD, CCV_KS1, CCV_TC>;

#define CCV_CAT2(a, b) a##b
#define CCV_CAT(a, b) CCV_CAT2(a, b)

CcVariant CCV_CAT(cc_variant_, CCV_NAME)() { return ccf::Launcher<VariantCfg>::variant(); }
