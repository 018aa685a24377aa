// (F, L) pairs served by the C-modes-per-lane kernel A (propagate_cml.cu): L lanes per trajectory, C = ceil(F / L) modes per
// lane, G = floor(32 / L) trajectories per warp.  Chosen for the smallest C / G (FP64 work per trajectory) among the splits
// whose state (4 C F doubles per lane) fits the 128 doubles of tensor memory a lane owns.  F <= 3 is served by the
// thread-per-trajectory kernels.  build.py compiles propagate_cml.cu once per row.
#pragma once
#define SCI_CML_FOR_EACH(X) X(4, 2) X(5, 2) X(6, 2) X(7, 4) X(8, 4) X(9, 3) X(10, 5) X(11, 6) X(12, 6)
