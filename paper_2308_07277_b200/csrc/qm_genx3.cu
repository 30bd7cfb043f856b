#define QM_GEN_TU 3
#include "qm_gen_tu.h"
