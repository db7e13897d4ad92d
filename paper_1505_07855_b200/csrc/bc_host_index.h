// Owner of the host transport arrays behind a bc_index_host* handed out by the library
// (bc_index_build_host, bc_index_build_gpu); released by bc_index_host_free.  Internal.
#pragma once
#include <stdint.h>

#include <vector>

#include "../../include/barracuda_b200.h"

struct BcBwtArrays {
    std::vector<uint64_t> bwt2;
    std::vector<uint32_t> occ;
};

struct BcHostIndexOwner {
    bc_index_host pub;                          // must be first: the public pointer is this object
    BcBwtArrays fwd, rev;
    std::vector<uint32_t> sa;
};
