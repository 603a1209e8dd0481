"""CPU: the roofline numerators bench.py uses - algorithmic bytes per drone and step of the five configs against
the table written out by hand from the data layout (§5), and the survey's flop tallies it quotes beside the oracle's."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2606_08039_b200 import workloads as W   # noqa: E402


def hand_bytes(c):
    """§5: planes are 16 B per drone.  Read: P0-P3 (64), target P6 (16), action row (16), + P4 (16) with an attitude loop, + P5
    (16) for PID.  Written: P0-P3 (64), P4 / P5 as read, the observation (12 floats, + M adjacency entries), the reward share (4).
    Per env: E0 + step counter read and written (2 x 20), reward (4), done (1)."""
    M = {1: 1, 2: 1, 3: 1, 4: 8, 5: 4}[c]
    if c in (1, 2, 4):                       # raw rotor commands
        per_drone = (64 + 16 + 16) + 64 + 48 + 4
    elif c == 3:                             # PID waypoints: P4 and P5 both ways
        per_drone = (64 + 16 + 16 + 32) + (64 + 32) + 48 + 4
    else:                                    # c5: VEL through the PID (P4 both ways), adjacency row of 4
        per_drone = (64 + 16 + 16 + 16) + (64 + 16) + (48 + 16) + 4
    return per_drone + (40 + 5) / M


@pytest.mark.parametrize("c", [1, 2, 3, 4, 5])
def test_algorithmic_bytes_match_the_layout(c):
    import bench
    assert bench.algorithmic_bytes_per_drone(W.config(c)) == pytest.approx(hand_bytes(c), abs=1e-9)
    # and DESIGN.md §6's table (rounded)
    assert round(bench.algorithmic_bytes_per_drone(W.config(c))) == {1: 257, 2: 257, 3: 321, 4: 218, 5: 271}[c]


def test_table4_planes_are_counted():
    import bench
    wl = W.config(5)
    base = bench.algorithmic_bytes_per_drone(wl)
    wl.params.update(W.VARIANTS["table4"])
    assert bench.algorithmic_bytes_per_drone(wl) - base == 64 + 32 + 96      # R0-R3 read, N0 both ways, H0-H2 both ways


def test_survey_tally_of_config_5():
    import bench
    assert bench.SURVEY_FLOPS_PER_DRONE_STEP[5] == 3540
