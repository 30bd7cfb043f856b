#define QM_TU_MODE 4
#include "qm_plane_tu.h"
