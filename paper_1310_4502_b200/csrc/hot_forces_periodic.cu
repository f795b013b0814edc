// Periodic (125-image) instantiations of the walk + interaction kernel, in their own translation
// unit so the two halves compile in parallel.  See hot_forces.cu.
#define HOT_FORCES_PERIODIC_TU 1
#include "hot_forces.cu"
