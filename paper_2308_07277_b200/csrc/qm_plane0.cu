#define QM_TU_MODE 0
#include "qm_plane_tu.h"
