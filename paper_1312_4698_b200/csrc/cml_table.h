// (F, L) pairs served by the C-modes-per-lane kernel A (propagate_cml.cu): L lanes per trajectory, C = ceil(F / L) modes per
// lane, G = floor(32 / L) trajectories per warp.  The state (4 C F doubles per lane) must fit the 128 doubles of tensor memory
// a lane owns.  L = 1 where it does (F = 4, 5: one lane per trajectory, no shuffles at all: 20.5 and 31.5 ms for 65536 x 4000
// trajectory-steps of the uncoupled Morse systems against 27.5 and 44.8 ms with L = 2); otherwise the fewest lanes that fit (F = 7,
// 8 with L = 2: 90.8 and 110.3 ms against 96.8 and 117.7 ms with L = 4; F = 10 with L = 4 or 5: the same), i.e. the most FMAs per
// shuffled pivot element.  Fractions of FP64 peak per row: profiles/r03_morse_sweep.md (Morse: 40 / 42 / 38 / 33 / 38 / 36 / 31 /
// 28 / 31 % for F = 4..12 with the flop that are executed; quartic force fields: 42.9 % at F = 6, 40.1 % at F = 9).
// F <= 3 is served by the thread-per-trajectory kernels.  build.py compiles propagate_cml.cu once per row.
#pragma once
#define SCI_CML_FOR_EACH(X) X(4, 1) X(5, 1) X(6, 2) X(7, 2) X(8, 2) X(9, 3) X(10, 5) X(11, 6) X(12, 6)
