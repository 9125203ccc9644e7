"""Digest an ncu report to the text summaries kept under profiles/.

    python -m paper_1208_2407_b200.ncu_digest report.ncu-rep > profiles/<name>.txt

Runs `ncu -i report --page raw --csv` (selected metrics per captured launch) and
`ncu -i report --page source --csv --print-source sass` (instruction mix weighted by executed
count, and the warp-stall sampling shares) and prints both as plain text.  Formatting only.
"""
import csv, subprocess, sys, collections
rep = sys.argv[1]
KEYS = ['gpu__time_duration.sum','dram__bytes_read.sum','dram__bytes_write.sum',
 'gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed','launch__registers_per_thread',
 'sm__warps_active.avg.pct_of_peak_sustained_active','launch__occupancy_limit_registers',
 'launch__occupancy_limit_shared_mem','smsp__inst_executed.sum',
 'sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active',
 'sm__inst_executed_pipe_lsu.avg.pct_of_peak_sustained_active',
 'sm__inst_executed_pipe_uniform.avg.pct_of_peak_sustained_active',
 'smsp__issue_active.avg.pct_of_peak_sustained_active','launch__grid_size',
 'launch__waves_per_multiprocessor','lts__t_sector_hit_rate.pct',
 'l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum','l1tex__data_pipe_lsu_wavefronts_mem_shared.sum',
 'launch__shared_mem_per_block_dynamic','sm__cycles_elapsed.avg.per_second']
out = subprocess.run(['ncu','-i',rep,'--page','raw','--csv'],capture_output=True,text=True).stdout
rows = list(csv.reader(out.splitlines()))
h, units = rows[0], rows[1]
for v in rows[2:]:
    d = dict(zip(h, v)); u = dict(zip(h, units))
    print('---', d.get('Kernel Name','')[:90], d.get('Grid Size',''), d.get('Block Size',''))
    for k in KEYS:
        if k in d: print(f'  {k:72s} {d[k]:>16s} {u[k]}')
src = subprocess.run(['ncu','-i',rep,'--page','source','--csv','--print-source','sass'],capture_output=True,text=True).stdout
kern = None; idx = -1
def flush(name, mix, stalls, total):
    if name is None: return
    print(f'=== kernel {idx} {name[:90]} warp instr {total}')
    tot = sum(mix.values()) or 1
    print('  mix: ' + ', '.join(f'{k} {100*v/tot:.1f}%' for k, v in mix.most_common(14)))
    ts = sum(stalls.values()) or 1
    print('  stalls: ' + ', '.join(f'{k} {100*v/ts:.1f}%' for k, v in stalls.most_common(9)))
mix = collections.Counter(); stalls = collections.Counter(); total = 0; hdr = None
for r in csv.reader(src.splitlines()):
    if not r: continue
    if r[0] == 'Kernel Name':
        flush(kern, mix, stalls, total)
        kern = r[1]; idx += 1; mix = collections.Counter(); stalls = collections.Counter(); total = 0; hdr = None
        continue
    if r[0] == 'Address': hdr = r; continue
    if hdr is None: continue
    d = dict(zip(hdr, r))
    op = d['Source'].split()
    if not op: continue
    o = op[1] if op[0].startswith('@') and len(op) > 1 else op[0]
    o = o.split('.')[0]
    n = int(d.get('Instructions Executed','0') or 0)
    mix[o] += n; total += n
    for k in hdr:
        if k.startswith('stall_') and 'Not Issued' not in k:
            stalls[k[6:]] += int(d.get(k,'0') or 0)
flush(kern, mix, stalls, total)
