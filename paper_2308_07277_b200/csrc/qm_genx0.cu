#define QM_GEN_TU 0
#include "qm_gen_tu.h"
