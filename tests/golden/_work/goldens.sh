#!/bin/bash
cd /root/repo/tests/golden
G="nice -n 10 python make_golden.py"
$G 1 1e7 > /root/repo/_work/g_cfg1.log 2>&1
$G 1 1e7 --coh 7e-30 > /root/repo/_work/g_cfg1c.log 2>&1
$G 2 1e6 > /root/repo/_work/g_cfg2.log 2>&1
$G 3 1e6 > /root/repo/_work/g_cfg3.log 2>&1
$G rays 1e6 > /root/repo/_work/g_rays.log 2>&1
$G 4 1e6 --nt 512 --bands 128 > /root/repo/_work/g_cfg4.log 2>&1
echo ALLDONE > /root/repo/_work/g_done.log
