"""The orientation table of k_node_solve (ZP_K3_ORIENT_MASK in csrc/kernels.cuh) is read off the SASS of one ptxas
version (python -m paper_2505_24256_b200.orient -> profiles/r02_k3_orient.md).  A different nvcc silently de-tunes
the 25 template instances: this test fails then, so that the table is derived again instead."""
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def recorded():
    txt = open(os.path.join(ROOT, "profiles", "r02_k3_orient.md")).read()
    return (re.search(r"^nvcc: (\S+)", txt, re.M).group(1), int(re.search(r"^derived mask: (0x[0-9a-f]+)", txt, re.M).group(1), 16),
            txt)


def test_nvcc_version_is_the_one_the_table_was_derived_with():
    from paper_2505_24256_b200 import orient

    ver, _, _ = recorded()
    assert orient.nvcc_version() == ver, ("nvcc changed: run `python -m paper_2505_24256_b200.orient --write "
                                          "profiles/r02_k3_orient.md` and update ZP_K3_ORIENT_MASK")


def test_mask_in_the_source_is_the_recorded_one():
    from paper_2505_24256_b200 import orient

    _, mask, txt = recorded()
    assert orient.current_mask() == mask
    # the mask is what the table says: bit NB set <=> order 1 chosen
    rows = re.findall(r"^\| (\d+) \| \d+ \| [\d.]+ \| \d+ \| [\d.]+ \| ([01]) \|", txt, re.M)
    assert len(rows) == 25 and sum(int(c) << int(nb) for nb, c in rows) == mask
