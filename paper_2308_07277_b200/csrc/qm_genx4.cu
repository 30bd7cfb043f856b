#define QM_GEN_TU 4
#include "qm_gen_tu.h"
