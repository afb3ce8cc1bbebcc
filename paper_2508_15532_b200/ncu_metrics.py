"""Turn an `ncu --page raw --csv` export of one rt_step into the per-kernel-class metrics bench.py quotes.

    python -m paper_2508_15532_b200.ncu_metrics <raw.csv> <config index> <out.json>

The output records the hash of the library sources it was captured from (`source_hash()`); bench.py reports
`roofline.traffic` and the other ncu-derived figures only when that hash equals the hash of the sources it runs, so a
number taken from another build can never be attached to a live time.  The capture command is written into the file.
"""
import csv
import glob
import hashlib
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)

# kernel name (substring) -> class of rt_profile_read
CLASSES = (("k_facecoef", "facecoef"), ("k_colflag", "facecoef"), ("k_transport", "transport"), ("k_angular", "angular"),
           ("k_cell", "source"), ("k_moments", "source"))
METRICS = {"dram_bytes": ("dram__bytes_read.sum", "dram__bytes_write.sum"), "warp_instr": ("smsp__inst_executed.sum",),
           "l2_to_l1_bytes": ("l1tex__m_xbar2l1tex_read_bytes.sum",), "time_us": ("gpu__time_duration.sum",)}
UNIT_SCALE = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "inst": 1.0, "us": 1.0, "ms": 1e3, "ns": 1e-3, "": 1.0}


def source_hash():
    """sha256 over the library's sources and its public header (what the .so is built from)."""
    h = hashlib.sha256()
    files = sorted(glob.glob(os.path.join(HERE, "csrc", "*"))) + [os.path.join(ROOT, "include", "rt.h")]
    for f in files:
        h.update(os.path.basename(f).encode())
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def summarise(raw_csv):
    rows = list(csv.reader(open(raw_csv)))
    hdr, units = rows[0], rows[1]
    iname = hdr.index("Kernel Name")
    out = {}
    for r in rows[2:]:
        cls = next((c for key, c in CLASSES if key in r[iname]), None)
        if cls is None:
            continue
        d = out.setdefault(cls, {"launches": 0, "kernels": {}})
        d["launches"] += 1
        short = r[iname].split("(")[0].split("::")[-1]
        d["kernels"][short] = d["kernels"].get(short, 0) + 1
        for key, cols in METRICS.items():
            for c in cols:
                if c in hdr:
                    i = hdr.index(c)
                    d[key] = d.get(key, 0.0) + float(r[i].replace(",", "")) * UNIT_SCALE.get(units[i], 1.0)
    return out


def main():
    raw, cfg, dst = sys.argv[1], int(sys.argv[2]), sys.argv[3]
    doc = {"source_hash": source_hash(), "config": cfg, "scope": "one rt_step (predictor + corrector), sums over the launches of a class",
           "command": "ncu --set full --clock-control none -k regex:^k_ -s <warm-up launches> -c <launches of one step> "
                      "python bench.py --config %d --steps 1 --warmup 3 --no-e2e --no-cpu-baseline; ncu -i <rep> --page raw --csv" % cfg,
           "classes": summarise(raw)}
    with open(dst, "w") as f:
        json.dump(doc, f, indent=1, sort_keys=True)
    print(json.dumps(doc["classes"], indent=1))


if __name__ == "__main__":
    main()
