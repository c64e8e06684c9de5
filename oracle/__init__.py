"""ORACLE (test infrastructure, NOT the product).  See ``oracle/ora.py`` and
``oracle/pic_oracle.h``.  Nothing under ``paper_2303_12873_b200`` imports this
package, and this package imports nothing from it."""
