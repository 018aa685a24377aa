// (F, L) pairs served by the C-modes-per-lane kernel A (propagate_cml.cu): L lanes per trajectory, C = ceil(F / L) modes per
// lane, G = floor(32 / L) trajectories per warp.  The state (4 C F doubles per lane) must fit the 128 doubles of tensor memory
// a lane owns.  L = 1 where it does (F = 4, 5: one lane per trajectory, no shuffles at all: 46 % and 51 % of FP64 peak on the
// uncoupled Morse systems against 34 % and 36 % with L = 2); otherwise the fewest lanes that fit (F = 7, 8 with L = 2: 42 % and 49 %
// against 39 % and 46 % with L = 4; F = 10 with L = 4 or 5: the same), i.e. the most FMAs per shuffled pivot element.
// F <= 3 is served by the thread-per-trajectory kernels.  build.py compiles propagate_cml.cu once per row.
#pragma once
#define SCI_CML_FOR_EACH(X) X(4, 1) X(5, 1) X(6, 2) X(7, 2) X(8, 2) X(9, 3) X(10, 5) X(11, 6) X(12, 6)
