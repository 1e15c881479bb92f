// RESIDENT engine placeholder (replaced by the register-resident persistent kernel).
#include "pimpc_internal.h"

bool resident_supported(const pimpc_s *, std::string *why)
{
    if (why) *why = "not built yet";
    return false;
}

int run_resident(pimpc_s *h, int, double)
{
    h->errmsg = "RESIDENT engine not available";
    return PIMPC_EINVAL;
}
