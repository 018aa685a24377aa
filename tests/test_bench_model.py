"""Host logic of bench.py that the roofline fraction rests on: the algorithmic flop model must reproduce SURVEY.md 8d's
table by hand, and the chirp-z plan must mirror the library's (csrc/api.cu chirp_plan)."""
import bench


def test_flop_model_is_the_survey_table():
    # SURVEY.md 8d, QFF rows: PES | 16F+6 | 2(2F^3+6F^2) | 6F^2 | complex det  (transcendentals are not kernel A's here)
    assert bench.flop_model(9, 4000, False)["propagate"] == 1386 + 150 + 3888 + 486 + 1980 == 7890
    assert bench.flop_model(9, 4000, True)["propagate"] == 7890 + 3570 == 11460
    assert bench.flop_model(6, 4000, False)["propagate"] == 528 + 102 + 1296 + 216 + 615
    assert bench.flop_model(6, 4000, True)["propagate"] == 528 + 102 + 1296 + 216 + 615 + 1012
    assert bench.flop_model(3, 4000, True)["propagate"] == 120 + 54 + 216 + 54 + 95 + 110
    assert bench.flop_model(1, 2000, True, morse=True)["propagate"] == 60 + 22 + 16 + 6 + 10 + 2
    # uncoupled Morse oscillators, F > 1: diagonal Hessian, so the monodromy column is 16 F^2 (= the F = 1 row's 16 at F = 1), not
    # the dense 2 (2 F^3 + 6 F^2) that the kernels never execute for them; the determinant columns stay dense
    assert bench.flop_model(5, 4000, True, morse=True)["propagate"] == 300 + 86 + 400 + 150 + (8 * 4 * 5 * 9 // 6 + 6 * 5 * 4 // 2 + 80) + 570
    assert bench.flop_model(9, 4000, True, morse=True)["propagate"] == 540 + 150 + 1296 + 486 + 1980 + 3570
    assert bench.flop_model(9, 4000, True)["propagate"] - bench.flop_model(9, 4000, True, morse=True)["propagate"] == (1386 - 540) + (3888 - 1296)
    # Fourier stage: direct sum 8k, chirp-z two FFTs of length 8192 per trajectory and block
    assert bench.flop_model(9, 4000, True, nblocks=0)["fourier"] == 32000
    one = bench.flop_model(9, 4000, True, nsteps=4000, nblocks=1)["fourier"]
    assert abs(one - 2 * 5 * 8192 * 13 / 4001) < 1e-9
    assert abs(bench.flop_model(9, 4000, True, nsteps=8000, nblocks=2)["fourier"] - 2 * 2 * 5 * 8192 * 13 / 8001) < 1e-9


def test_chirp_plan_mirror():
    assert bench.chirp_blocks(4000, 4000) == 1          # 8000 <= 8192: one block
    assert bench.chirp_blocks(8000, 4000) == 2          # blocks of 8193 - 4000 = 4193 samples
    assert bench.chirp_blocks(3000, 2000) == 1
    assert bench.chirp_blocks(4000, 7500) == 0          # block shorter than 1024: direct sum
    assert bench.chirp_blocks(100000, 4000) == 0        # more than 16 blocks: direct sum
