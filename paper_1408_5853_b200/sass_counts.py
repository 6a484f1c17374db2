"""Static SASS mnemonic counts per compiled kernel of libheat_b200.so (profiles/r02_sass_counts.txt):

    cuobjdump -sass paper_1408_5853_b200/libheat_b200.so | python -m paper_1408_5853_b200.sass_counts

UTMALDG/UTMASTG = cp.async.bulk.tensor (TMA) load/store, UBLKCP = cp.async.bulk, SYNCS = mbarrier ops,
STAS = st.async, LDTM/STTM = tcgen05.ld/st (tensor memory), UTCATOMSWS = tcgen05.alloc, UCGABAR = cluster barrier.
"""
import re
import subprocess
import sys

MN = ["UTMALDG", "UTMASTG", "UBLKCP", "SYNCS", "STAS", "LDTM", "STTM", "UTCATOMSWS", "DFMA", "DMUL", "DADD",
      "MUFU.RCP64H", "MUFU.RSQ64H", "SHFL", "BAR.SYNC", "UCGABAR"]


def main():
    pat = re.compile(r"^\s+/\*[0-9a-f]{4,}\*/\s+(?:@!?U?P\d\s+)?([A-Z0-9_.]+)")
    rows, cur = [], None
    for line in sys.stdin:
        if line.lstrip().startswith("Function :"):
            if cur:
                rows.append(cur)
            cur = {"name": line.split(":", 1)[1].strip(), "total": 0, **{m: 0 for m in MN}}
            continue
        m = pat.match(line)
        if m and cur is not None:
            op = m.group(1)
            cur["total"] += 1
            for k in MN:
                if op == k or op.startswith(k + "."):
                    cur[k] += 1
    if cur:
        rows.append(cur)
    names = subprocess.run(["c++filt"], input="\n".join(r["name"] for r in rows), capture_output=True, text=True).stdout.splitlines()
    print("kernel | total | " + " | ".join(MN))
    for r, d in zip(rows, names):
        d = re.sub(r"^void heat::|\(heat::\w+\)$", "", d).replace("(int)", "")
        print(d + " | " + str(r["total"]) + " | " + " | ".join(str(r[k]) for k in MN))


if __name__ == "__main__":
    main()
