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
