// Dynamic, in-order tile scheduling for the persistent contraction kernel (K2).
//
// With a static assignment (CTA pair g takes tiles g, g + G, g + 2G, ...) nothing keeps the pairs
// in step: small speed differences between SMs accumulate over the ~440 tiles of a pair, the set
// of tiles in flight spreads over many channels / row blocks, and the sharing of operand blocks
// through L2 collapses (measured at N = 4096: 41-58 GB instead of 9 GB of DRAM reads per launch).
// Handing the tiles out in index order from one global counter -- as the hardware block scheduler
// would, but to persistent CTAs -- keeps the window of tiles in flight compact.  Every tile is
// computed the same way whichever pair gets it, so results stay bitwise reproducible.
//
// The scheduler words live in a pool in global memory ({next tile, drained CTA groups} per
// launch); the last group to run dry re-arms its pair for a later launch (k2_contract.cu).
// K1 / K3 keep the static assignment: their tiles share nothing, and the same scheduler measured
// no gain there.
#pragma once

namespace foldcp {

// host side (api.cu): a pair of zeroed scheduler words for one launch; nullptr on CUDA error
unsigned int* next_sched_slot();

}  // namespace foldcp
