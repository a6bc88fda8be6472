"""Front end: BED parsing, half-open -> closed conversion, projection.  No GPU."""
import numpy as np
import pytest

from paper_1208_3407_b200 import frontend as F


def _write(tmp_path, name, text):
    p = tmp_path / name
    p.write_text(text)
    return str(p)


def test_genome_and_projection(tmp_path):
    g = F.read_genome(_write(tmp_path, "g.txt", "# a comment\nchr1 1000\nchr2\t500\n\nchrX 250\n"))
    assert g.names == ["chr1", "chr2", "chrX"] and g.offsets.tolist() == [0, 1000, 1500, 1750]
    bed = "track name=x\nchr1\t0\t10\tfeature\nchr2 5 6\n#skip\nchrX\t249\t250\t.\t0\t+\nchr1 990 1000\n"
    s, e = F.read_bed(_write(tmp_path, "a.bed", bed), g)
    # half-open [s, e) on the chromosome -> closed [off + s, off + e - 1]
    assert s.tolist() == [0, 1005, 1749, 990] and e.tolist() == [9, 1005, 1749, 999]
    assert s.dtype == np.uint32 and e.dtype == np.uint32


def test_adjacent_bed_intervals_do_not_touch_after_conversion(tmp_path):
    """[0,10) and [10,20) share no base: closed [0,9] and [10,19] (the closed rule of PAPER.md:31 would count a shared end point)."""
    g = F.read_genome(_write(tmp_path, "g.txt", "c 100\n"))
    s, e = F.read_bed(_write(tmp_path, "a.bed", "c 0 10\nc 10 20\n"), g)
    assert e[0] < s[1]


@pytest.mark.parametrize("bed,msg", [("chr9 1 2\n", "not in the genome"), ("chr1 5 5\n", "start < end"), ("chr1 0 1001\n", "start < end"),
                                      ("chr1 x 3\n", "integers"), ("chr1 4\n", "needs chrom")])
def test_bad_bed_lines(tmp_path, bed, msg):
    g = F.read_genome(_write(tmp_path, "g.txt", "chr1 1000\n"))
    with pytest.raises(F.FrontEndError, match=msg):
        F.read_bed(_write(tmp_path, "a.bed", bed), g)


def test_skip_unknown_and_bad_genomes(tmp_path):
    g = F.read_genome(_write(tmp_path, "g.txt", "chr1 1000\n"))
    s, e = F.read_bed(_write(tmp_path, "a.bed", "chrUn 1 2\nchr1 1 2\n"), g, skip_unknown=True)
    assert s.tolist() == [1] and e.tolist() == [1]
    for text in ("", "chr1 0\n", "chr1 10\nchr1 20\n", "chr1 4294967296\n"):
        with pytest.raises(F.FrontEndError):
            F.read_genome(_write(tmp_path, "bad.txt", text))
