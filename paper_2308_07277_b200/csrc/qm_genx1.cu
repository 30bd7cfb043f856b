#define QM_GEN_TU 1
#include "qm_gen_tu.h"
