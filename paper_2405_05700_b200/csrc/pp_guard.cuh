// Device-side invariant checks of the test-only guard build (-DPP_GUARD; tests/test_gpu_guard.py), standing in for
// compute-sanitizer's memcheck on the propagation kernel's index arithmetic (the pool's wrapper
// refuses that tool).  In the product build PP_GUARD_CHECK compiles to nothing.  A failed check stores its code in
// Status::error (first one wins), which the host reports as "internal: ..." after the launch; the access it guards is
// then skipped by the caller where the macro's value is used.
#pragma once

#ifdef PP_GUARD
#define PP_GUARD_CHECK(st, cond, code) ((cond) ? true : (atomicCAS(&(st)->error, 0u, (unsigned)(code)), false))
#else
#define PP_GUARD_CHECK(st, cond, code) (true)
#endif

// codes (Status::error; 1 = resume list overflow, set by the product build too)
#define PP_GUARD_SRC_INDEX 16   // a warp's current source index ran past n_src
#define PP_GUARD_TILE_SRC 17    // a tile's first source index is not below n_src
#define PP_GUARD_FATE_INDEX 18  // a fate record would land outside [0, g_end)
#define PP_GUARD_HIT_SLOT 19    // a hit would be stored at or beyond ring_cap
#define PP_GUARD_RESUME_SLOT 20 // a resume item would be stored at or beyond resume_cap
#define PP_GUARD_PHOTON_INDEX 21 // a photon index is not below its source's photon count
