cd _work
for b in ub_*; do [ -x $b ] && ./$b 65536; done
